// rsos_resident.cu -- the RESIDENT engine: DT schedule on lattices small enough to live on chip (sm_100a).
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// BASELINE.json north_star (3) / P:75: "a whole lattice lives on-chip for many sweeps".  When a
// colour pass of the DT schedule (D:2 steps 4-6) has only a few tiles per realization (L = 128
// ... 512 at S = 64: 1, 4, 16), one kernel launch per pass re-stages every tile from global memory 4K
// times per MCS and the machine waits on launches.  Here a thread block -- or a CLUSTER of C thread
// blocks that share their shared memory (DSMEM) -- owns one realization for ALL colour passes,
// sub-sweeps and MCS of an rsos_advance call:
//   * the lattice lives in shared memory with one element per site (uint8 when the packed HBM lattice
//     has 2-bit sites, uint16 with 4-bit sites, D:5): low FB bits = height mod 2^FB, next 5 bits = the
//     lane that last wrote the site.  Block c of the cluster holds rows [c L/C, (c+1) L/C); a row has a
//     pitch of one word more than its length, so 32 lanes copying 32 different rows hit 32 banks;
//   * per pass a warp copies its tile window (S + 2)^2 out of the resident lattice (possibly from the
//     other blocks of the cluster), runs the S*S/K attempts of the tile, and copies the S x S interior
//     back; one block / cluster barrier per pass;
//   * one warp per tile, 32 consecutive attempts in flight (D:4, the window step of the WARP engine in
//     its cheapest form): every lane loads its 5-point stencil (5 element loads at immediate offsets),
//     decides on that snapshot, accepting lanes store (height + 1, lane tag), every lane loads the
//     stencil again.  A lane is DIRTY if its own store is not what the site now holds, or its site or
//     a neighbour was written by a LOWER lane (the tag says who).  With f = lowest dirty lane, lanes
//     < f are final, accepting lanes >= f take their store back, and the next window starts at
//     attempt a0 + f.  Lane 0 depends on nothing, so f >= 1.  Two attempts interact only through equal
//     or adjacent sites, so the committed prefix is exactly the sequential result (checked bit for bit
//     against the oracle, tests/test_gpu_parity.py);
//   * the 16-bit Philox slots (D:2 step 6) of 256 attempts at a time go through a shared-memory table:
//     one 128-bit store per lane and 256 attempts, one 16-bit load per lane and window.
#include <cooperative_groups.h>

#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace cg = cooperative_groups;

namespace rsos {

template <int LGS, int FB>
struct RGeom {
    static constexpr uint32_t S = 1u << LGS;
    static constexpr uint32_t VM = (1u << FB) - 1u;               // height bits of an on-chip site (one byte per site)
    static constexpr uint32_t TS = FB == 2 ? 0u : 1u;             // tag = lane >> TS sits above the height bits
    static constexpr uint32_t PWW = (S + 2u + 3u) / 4u;           // words per window row
    static constexpr uint32_t WINW = PWW * (S + 2u);              // words per window
    static constexpr uint32_t ROWB = PWW * 4u;                    // bytes per window row
};

struct ResidentShape {
    uint32_t tpp;          // tiles per colour pass of one realization = (L / 2S)^2
    uint32_t csize;        // blocks per cluster (1 = no cluster)
    uint32_t warps;        // warps per block = tpp / csize
    uint32_t rows;         // lattice rows per block = L / csize
    uint32_t lgrows;
    uint32_t aligned;      // 1: a block takes the tiles whose first row lies in its slab (csize <= L / 2S)
};

__device__ __forceinline__ uint32_t lds_u8(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_u8(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u8 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void sts_v4(uint32_t addr, const uint4 &c)
{
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(c.x), "r"(c.y), "r"(c.z), "r"(c.w) : "memory");
}

// A chunk of the packed HBM lattice that holds 4 sites (8 bits at FB = 2, 16 bits at FB = 4) -> 4 bytes, and back
// (height bits only: the tags are dropped).
template <int FB> __device__ __forceinline__ uint32_t spread4(uint32_t o);
template <> __device__ __forceinline__ uint32_t spread4<2>(uint32_t o)
{
    uint32_t t = (o | (o << 12)) & 0x000F000Fu;
    return (t | (t << 6)) & 0x03030303u;
}
template <> __device__ __forceinline__ uint32_t spread4<4>(uint32_t o)
{
    uint32_t t = (o | (o << 8)) & 0x00FF00FFu;
    return (t | (t << 4)) & 0x0F0F0F0Fu;
}
template <int FB> __device__ __forceinline__ uint32_t gather4(uint32_t w);
template <> __device__ __forceinline__ uint32_t gather4<2>(uint32_t w)
{
    uint32_t t = w & 0x03030303u;
    t = (t | (t >> 6)) & 0x000F000Fu;
    return (t | (t >> 12)) & 0xFFu;
}
template <> __device__ __forceinline__ uint32_t gather4<4>(uint32_t w)
{
    uint32_t t = w & 0x0F0F0F0Fu;
    t = (t | (t >> 4)) & 0x00FF00FFu;
    return (t | (t >> 8)) & 0xFFFFu;
}

// One window of 32 attempts: lane = rank, attempt a0 + lane.
struct Win {
    uint32_t aC;                 // shared-memory address of the lane's site
    uint32_t c, l, r, u, d;      // snapshot of the 5-point stencil (whole bytes: height and tag)
    uint32_t W;                  // what an accepting lane stores
    bool valid, acc, dup;        // attempt exists; accepted on the snapshot; (4-bit sites) my pair partner accepted the same site
};

// One block = the rows [crank * rows, (crank + 1) * rows) of one realization and tpp / csize of its tiles.
// Shared memory: [rows x (L / 4 + 1) words: lattice slab][per warp: 256 words of slots][per warp: window].
template <int LGS, int FB, bool CLUSTER>
__global__ void __launch_bounds__(512) resident_dt_kernel(Params p, uint32_t t0, uint32_t mcs, ResidentShape sh)
{
    using G = RGeom<LGS, FB>;
    constexpr uint32_t S = G::S, PWW = G::PWW, VM = G::VM, ROWB = G::ROWB, TS = G::TS;
    constexpr uint32_t FULL = 0xFFFFFFFFu;
    extern __shared__ __align__(16) uint32_t smem[];
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t L = p.L, Lm = L - 1u;
    const uint32_t LW = L >> 2, LWm = LW - 1u, LP = LW + 1u;             // lattice row: words, mask, pitch
    const uint32_t T = L >> LGS, half = T >> 1;
    uint32_t crank = 0;
    if (CLUSTER) crank = cg::this_cluster().block_rank();
    const uint32_t rl = CLUSTER ? blockIdx.x / sh.csize : blockIdx.x;    // realization (local index)
    const uint32_t rg = p.first_real + rl;

    uint32_t *lat = smem;                                                 // my slab
    uint32_t *tab = smem + sh.rows * LP + warp * 256u;                    // 16-byte aligned: rows * LP is a multiple of 4 words
    uint32_t *win = smem + sh.rows * LP + sh.warps * 256u + warp * G::WINW;
    const uint32_t winb = (uint32_t)__cvta_generic_to_shared(win);
    const uint32_t tabb = (uint32_t)__cvta_generic_to_shared(tab);

    // ---- load my slab: packed HBM words (FB bits per site) -> one byte per site ------------------------------
    const uint32_t wpr = L >> (FB == 2 ? 4 : 3);                         // packed words per lattice row
    constexpr uint32_t WPP = FB == 2 ? 4u : 2u;                           // on-chip words per packed word
    const uint32_t *pk = p.pk + (size_t)rl * L * wpr + (size_t)crank * sh.rows * wpr;
    for (uint32_t i = tid; i < sh.rows * wpr; i += blockDim.x) {
        const uint32_t yl = i / wpr, w = i - yl * wpr;
        const uint32_t v = pk[i];
        uint32_t *dst = lat + yl * LP + WPP * w;
#pragma unroll
        for (uint32_t q = 0; q < WPP; ++q) dst[q] = spread4<FB>((v >> ((32u / WPP) * q)) & ((1u << (32u / WPP)) - 1u));
    }
    if (CLUSTER) cg::this_cluster().sync(); else __syncthreads();

    const uint32_t A = (S * S) / p.K;
    const uint32_t N = p.N;
    uint32_t nacc = 0;

    auto slot = [&](uint32_t a) -> uint32_t { return lds_u16(tabb + ((a & 511u) << 1)); };
    auto site = [&](uint32_t v) -> uint32_t {                            // D:2 step 6: dx = v & (S-1), dy = (v >> lg S) & (S-1)
        return winb + (((v >> LGS) & (S - 1u)) + 1u) * ROWB + (v & (S - 1u)) + 1u;
    };
    auto load5 = [&](uint32_t aC, uint32_t &c, uint32_t &l, uint32_t &r, uint32_t &u, uint32_t &d) {
        c = lds_u8(aC); l = lds_u8(aC - 1u); r = lds_u8(aC + 1u); u = lds_u8(aC - ROWB); d = lds_u8(aC + ROWB);
    };
    // Eq. (6) under the invariant |dh| <= N: rejected iff some neighbour sits at h - N (mod 2^FB)
    auto decide = [&](Win &w, bool valid) {
        const uint32_t tq = w.c - N;
        const uint32_t hit = ((w.l ^ tq) & VM) * ((w.r ^ tq) & VM) * ((w.u ^ tq) & VM) * ((w.d ^ tq) & VM);   // 0 iff some neighbour blocks
        w.valid = valid;
        w.acc = valid & (hit != 0u);
        w.W = ((w.c + 1u) & VM) | ((lane >> TS) << FB);
        w.dup = false;
        if (TS) {                                                         // two lanes share a tag: the odd one checks its partner
            const uint32_t pa = __shfl_xor_sync(FULL, w.acc ? w.aC : 0u, 1);
            w.dup = w.acc & (pa == w.aC) & ((lane & 1u) != 0u);
        }
    };

    for (uint32_t m = 0; m < mcs; ++m)
    for (uint32_t k = 0; k < p.K; ++k) {
        const uint32_t u = (t0 + m) * p.K + k;
        uint32_t ox, oy;
        draw_origin(p, u, rg, ox, oy);
#pragma unroll 1
        for (uint32_t colour = 0; colour < 4; ++colour) {
            // my tile of this pass: fixed share, or (aligned) the tiles whose first row lies in my slab
            uint32_t ti, tj;
            if (sh.aligned) {
                const uint32_t base = (oy + (colour >> 1) * S) & Lm;      // first row of tile row tj = 0
                const uint32_t dist = (crank * sh.rows - base) & Lm;
                ti = warp % half;
                tj = (((dist + 2u * S - 1u) >> (LGS + 1)) + warp / half) & (half - 1u);
            } else {
                const uint32_t n = crank * sh.warps + warp;
                ti = n % half; tj = n / half;
            }
            const uint32_t I = 2 * ti + (colour & 1u), J = 2 * tj + (colour >> 1);
            const uint32_t x0 = (ox + I * S) & Lm, y0 = (oy + J * S) & Lm;
            const uint32_t tile_id = J * T + I;

            // slots of attempts 0 .. 511: lane l computes Philox calls l and 32 + l (D:2 step 6)
            sts_v4(tabb + lane * 16u, philox4x32_10(lane, tile_id, u, rg, p.k0, p.k1));
            if (A > 256u) sts_v4(tabb + 512u + lane * 16u, philox4x32_10(32u + lane, tile_id, u, rg, p.k0, p.k1));

            // ---- a3: window rows y0-1 .. y0+S, columns x0-1 .. x0+S, out of the resident lattice --------------
            {
                const uint32_t sx = (x0 - 1u) & Lm;
                const uint32_t w0 = sx >> 2, ob = (sx & 3u) * 8u;
#pragma unroll 1
                for (uint32_t yr = lane; yr < S + 2u; yr += 32u) {
                    const uint32_t y = (y0 - 1u + yr) & Lm;
                    const uint32_t owner = y >> sh.lgrows, yl = y & (sh.rows - 1u);
                    const uint32_t *rowp = lat + yl * LP;
                    if (CLUSTER && owner != crank) rowp = cg::this_cluster().map_shared_rank(lat, owner) + yl * LP;
                    uint32_t prev = rowp[w0 & LWm];
                    uint32_t *wr = win + yr * PWW;
#pragma unroll
                    for (uint32_t q = 0; q < PWW; ++q) {
                        const uint32_t nxt = rowp[(w0 + q + 1u) & LWm];
                        wr[q] = __funnelshift_r(prev, nxt, ob);
                        prev = nxt;
                    }
                }
            }
            __syncwarp();

            // ---- a1 + a4: the A attempts of the tile, 32 at a time, exactly as if one after another.  The reload that
            // verifies window k and the snapshot of window k + 1 (which is valid if k turns out clean, the common
            // case) are issued together, so a clean window costs one shared-memory round trip. ----------------------
            uint32_t a0 = 0;
            Win cur, nxt;
            bool cold = true;
#pragma unroll 1
            while (a0 < A) {
                if (cold) {                                               // start (or restart after a partial commit) at a0
                    cur.aC = site(slot(a0 + lane));
                    load5(cur.aC, cur.c, cur.l, cur.r, cur.u, cur.d);
                    nxt.aC = site(slot(a0 + 32u + lane));
                    decide(cur, a0 + lane < A);
                    __syncwarp();
                    if (cur.acc) sts_u8(cur.aC, cur.W);
                    __syncwarp();
                    cold = false;
                }
                uint32_t c2, l2, r2, u2, d2;
                load5(cur.aC, c2, l2, r2, u2, d2);
                load5(nxt.aC, nxt.c, nxt.l, nxt.r, nxt.u, nxt.d);
                const uint32_t vnn = slot(a0 + 64u + lane);
                const uint32_t want = cur.acc ? cur.W : cur.c;
                const uint32_t diff = ((c2 ^ want) | (l2 ^ cur.l)) | ((r2 ^ cur.r) | (u2 ^ cur.u)) | (d2 ^ cur.d);
                decide(nxt, a0 + 32u + lane < A);
                uint32_t f = 32u;
                uint32_t bal = __ballot_sync(FULL, cur.valid & ((diff != 0u) | cur.dup));
                if (bal) {
                    // who wrote?  A write by a HIGHER lane cannot affect my decision.  (If a lower and a higher lane both
                    // wrote a site and the higher one's store is what remains, the lower one sees its own store gone.)
                    auto lower = [&](uint32_t now, uint32_t before) -> bool { return (now != before) & ((((now >> FB) << TS) & 31u) < lane); };
                    const bool dirty = cur.valid & ((cur.acc ? ((c2 != cur.W) | cur.dup) : lower(c2, cur.c)) | lower(l2, cur.l) |
                                                    lower(r2, cur.r) | lower(u2, cur.u) | lower(d2, cur.d));
                    bal = __ballot_sync(FULL, dirty);
                    if (bal) {
                        f = (uint32_t)__ffs((int)bal) - 1u;
                        if (f == 0u) f = 1u;                              // lane 0 stands whatever happened around it
                        // take back a store that is still there (a dup lane's byte equals its partner's: the partner decides)
                        if (cur.acc & !cur.dup & (lane >= f) & (c2 == cur.W)) sts_u8(cur.aC, cur.c);
                        __syncwarp();
                        if (cur.acc & (lane == 0u)) sts_u8(cur.aC, cur.W); // ... which may have hidden lane 0's
                        __syncwarp();
                        cold = true;
                    }
                }
                nacc += (cur.acc & (lane < f)) ? 1u : 0u;
                const uint32_t a1 = a0 + f;
                if ((a1 >> 8) != (a0 >> 8)) {
                    // entering block b = a1 >> 8 of 256 attempts: block b + 1 replaces block b - 1 in the table
                    const uint32_t b1 = (a1 >> 8) + 1u;
                    if (b1 * 256u < A) sts_v4(tabb + (b1 & 1u) * 512u + lane * 16u, philox4x32_10(32u * b1 + lane, tile_id, u, rg, p.k0, p.k1));
                    __syncwarp();
                }
                a0 = a1;
                if (!cold) {                                              // window k + 1 becomes the current one
                    cur = nxt;
                    nxt.aC = site(vnn);
                    __syncwarp();
                    if (cur.acc) sts_u8(cur.aC, cur.W);
                    __syncwarp();
                }
            }
            __syncwarp();

            // ---- a5: the S x S interior back into the resident lattice.  Lattice word j of a tile row holds the
            // window bits starting at 32 j - db + 8; the (at most two) partial edge words are merged with a plain
            // read-modify-write: no other tile of this pass touches them (tiles of a colour are 2S apart).
            {
                const uint32_t dw0 = x0 >> 2, db = (x0 & 3u) * 8u;
                constexpr uint32_t NWF = S / 4u;                          // words of an aligned tile row
                const bool neg = db > 8u;                                 // window bit offset 8 - db < 0
                const uint32_t sh_r = (8u - db) & 31u;
                const uint32_t first_mask = FULL << db;
#pragma unroll 1
                for (uint32_t yr = 1u + lane; yr <= S; yr += 32u) {
                    const uint32_t y = (y0 - 1u + yr) & Lm;
                    const uint32_t owner = y >> sh.lgrows, yl = y & (sh.rows - 1u);
                    uint32_t *rowp = lat + yl * LP;
                    if (CLUSTER && owner != crank) rowp = cg::this_cluster().map_shared_rank(lat, owner) + yl * LP;
                    const uint32_t *wr = win + yr * PWW;
                    uint32_t wv[NWF + 2];                                 // wv[i] = window word i - 1 (0 for i = 0)
                    wv[0] = 0u;
#pragma unroll
                    for (uint32_t i = 0; i <= NWF; ++i) wv[i + 1] = wr[i];
#pragma unroll
                    for (uint32_t j = 0; j <= NWF; ++j) {
                        const uint32_t lo = neg ? wv[j] : wv[j + 1];
                        const uint32_t hi = neg ? wv[j + 1] : (j < NWF ? wv[j < NWF ? j + 2 : 0] : 0u);
                        const uint32_t val = __funnelshift_r(lo, hi, sh_r);
                        uint32_t *dst = rowp + ((dw0 + j) & LWm);
                        if (j == 0u) { if (db) *dst = (*dst & ~first_mask) | (val & first_mask); else *dst = val; }
                        else if (j == NWF) { if (db) *dst = (*dst & first_mask) | (val & ~first_mask); }
                        else *dst = val;
                    }
                }
            }
            if (CLUSTER) cg::this_cluster().sync(); else __syncthreads();   // the next pass reads what this one wrote
        }
    }

    // ---- store my slab (height bits only), add the accepted counts --------------------------------------------
    {
        uint32_t *pko = p.pk + (size_t)rl * L * wpr + (size_t)crank * sh.rows * wpr;
        for (uint32_t i = tid; i < sh.rows * wpr; i += blockDim.x) {
            const uint32_t yl = i / wpr, w = i - yl * wpr;
            const uint32_t *src = lat + yl * LP + WPP * w;
            uint32_t v = 0;
#pragma unroll
            for (uint32_t q = 0; q < WPP; ++q) v |= gather4<FB>(src[q]) << ((32u / WPP) * q);
            pko[i] = v;
        }
    }
    // A launch covers up to 2^36 attempts (rsos_api.cu) and a warp may own all of them (one tile per colour pass, R = 1):
    // a lane's count stays below 2^31, the warp's total does not fit 32 bits -- sum the lanes in 64.
    unsigned long long tot = nacc;
#pragma unroll
    for (int o = 16; o; o >>= 1) tot += __shfl_xor_sync(FULL, tot, o);
    if (lane == 0 && tot) atomicAdd(p.accepted + rl, tot);
}

// =============================================================================================
// Host side
// =============================================================================================
static bool shape_of(uint32_t L, uint32_t lgS, uint32_t csize, ResidentShape *sh)
{
    const uint32_t half = (L >> lgS) >> 1;
    sh->tpp = half * half;
    sh->csize = csize;
    if (sh->tpp > 16u * csize || sh->tpp % csize || L % csize) return false;   // at most 16 warps per block
    sh->warps = sh->tpp / csize;
    sh->rows = L / csize;
    sh->lgrows = 0;
    while ((1u << sh->lgrows) < sh->rows) ++sh->lgrows;
    // whole tile rows per slab: every block can take the tiles that start in its own rows (mostly local copies)
    sh->aligned = (csize > 1 && csize <= half) ? 1u : 0u;
    return (1u << sh->lgrows) == sh->rows;
}

template <int LGS, int FB>
static size_t smem_of(uint32_t L, const ResidentShape &sh)
{
    using G = RGeom<LGS, FB>;
    return ((size_t)sh.rows * (L / 4 + 1) + (size_t)sh.warps * 256 + (size_t)sh.warps * G::WINW) * 4;
}

// what: 0 = shared-memory bytes (*out), 1 = set the function attributes, 2 = launch
template <int LGS, int FB, bool CLUSTER>
static cudaError_t resident_t(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st, int what, size_t *out)
{
    ResidentShape sh;
    if (!shape_of(p.L, p.lgS, p.CS, &sh)) return cudaErrorInvalidValue;
    const size_t sm = smem_of<LGS, FB>(p.L, sh);
    if (what == 0) { *out = sm; return cudaSuccess; }
    auto kern = resident_dt_kernel<LGS, FB, CLUSTER>;
    if (what == 1) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        if (e == cudaSuccess && sh.csize > 8) e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.R * sh.csize);
    cfg.blockDim = dim3(sh.warps * 32);
    cfg.dynamicSmemBytes = sm;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = sh.csize; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = CLUSTER ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, p, t0, mcs, sh);
}

template <int LGS, int FB>
static cudaError_t resident_k(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st, int what, size_t *out)
{
    return p.CS > 1 ? resident_t<LGS, FB, true>(p, t0, mcs, st, what, out) : resident_t<LGS, FB, false>(p, t0, mcs, st, what, out);
}

static cudaError_t resident_dispatch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st, int what, size_t *out)
{
    const bool two = p.FB == 2;
    switch (p.lgS) {
        case 4: return two ? resident_k<4, 2>(p, t0, mcs, st, what, out) : resident_k<4, 4>(p, t0, mcs, st, what, out);
        case 5: return two ? resident_k<5, 2>(p, t0, mcs, st, what, out) : resident_k<5, 4>(p, t0, mcs, st, what, out);
        case 6: return two ? resident_k<6, 2>(p, t0, mcs, st, what, out) : resident_k<6, 4>(p, t0, mcs, st, what, out);
        default: return cudaErrorInvalidValue;
    }
}

// Can the RESIDENT engine run (L, N, S, K) with clusters of `csize` blocks within smem_limit bytes per block?
// Needs DT mode, 16 <= S <= 64, N <= 7, tile^2 / K >= 32, csize in {1, 2, 4, 8, 16} dividing the tiles of a pass,
// at most 16 warps per block, and the lattice slab plus windows in shared memory.
bool resident_ok(uint32_t L, uint32_t N, uint32_t S, uint32_t K, uint32_t csize, size_t smem_limit)
{
    if (S < 16 || S > 64 || N > 7 || 2 * S > L || L > 65536) return false;
    if (csize != 1 && csize != 2 && csize != 4 && csize != 8 && csize != 16) return false;
    if (S * S / K < 32) return false;
    Params p{};
    p.L = L; p.lgS = S == 16 ? 4 : S == 32 ? 5 : 6; p.FB = thread_dt_field_bits(N, S); p.CS = csize;
    ResidentShape sh;
    if (!shape_of(L, p.lgS, csize, &sh)) return false;
    size_t sm = 0;
    if (resident_dispatch(p, 0, 0, nullptr, 0, &sm) != cudaSuccess) return false;
    return sm <= smem_limit;
}

// Cluster size the library picks: the smallest one whose slab fits the shared memory of a block (copies between
// blocks of a cluster go through DSMEM and cost more than local ones; a cluster barrier costs more than a block's).
uint32_t resident_cluster_size(uint32_t L, uint32_t N, uint32_t S, uint32_t K, uint32_t R, int sm_count, size_t smem_limit)
{
    (void)R; (void)sm_count;
    for (uint32_t k = 1; k <= 8; k *= 2) if (resident_ok(L, N, S, K, k, smem_limit)) return k;
    return 0;
}

size_t resident_smem(const Params &p)
{
    size_t sm = 0;
    resident_dispatch(p, 0, 0, nullptr, 0, &sm);
    return sm;
}

cudaError_t resident_configure(const Params &p) { return resident_dispatch(p, 0, 0, nullptr, 1, nullptr); }

uint32_t resident_blocks(const Params &p) { return p.R * p.CS; }

// `mcs` whole MCS starting at sweep counter t0, all colour passes and sub-sweeps inside one launch.
cudaError_t resident_launch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st)
{
    return resident_dispatch(p, t0, mcs, st, 2, nullptr);
}

}  // namespace rsos
