// rsos_gthread.cu -- the lane-per-tile engine on the packed lattice for lattice sides that are NOT powers of two (sm_100a).
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// The general-L schedule DTG(64, K) of D:2b (the paper's L = 9605; "a subset of domains have larger lateral size",
// P:204): T = 2 floor(L / 128) tiles per side with edges floor(i L / T), i.e. tiles of w x hgt sites, w, hgt in
// {floor(L / T), ceil(L / T)}.  When ceil(L / T) <= 66 a tile window of (w + 2) x (hgt + 2) sites still fits the row pitch
// of the THREAD engine's windows (PW words: 80 two-bit or 72 four-bit sites), so the same machinery applies (D:4, D:5):
//   * working state = the packed lattice, FB bits per site (height mod 2^FB), row pitch ceil(L FB / 32) words
//     (rsos_pack.cu, general kernels); the int32 heights are rebuilt on demand;
//   * one lane per tile, 32 tiles per warp, windows word-interleaved in shared memory (word w of tile g at
//     smem[w * 32 + g]): every shared-memory access of the attempt loop is conflict-free;
//   * the attempt is Attempt<6, FB, 1> (rsos_attempt.cuh): fields compared in the top bits, whole-word store.
// What differs from thread_dt_kernel: the site comes from the exactly uniform bounded draw of the tile's Philox word
// stream (s = draw(w hgt), dx = s mod w, dy = s div w), the origin from draw(L) twice, and a lattice row is a periodic
// string of L FB bits that does not end on a word boundary, so staging and write-back move bit ranges:
// get_bits() reads 32 bits at any bit position of the periodic row, put_range() writes a bit range word by word
// (whole words stored, partial words merged with atomicAnd / atomicOr; tiles of one colour are >= 64 sites apart, so
// no other tile of the pass owns bits of those words).
#include "rsos_attempt.cuh"
#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace rsos {

// 32 bits of the periodic bit string of one packed lattice row (LB = L * FB bits in wpr words) starting at bit b < LB
__device__ __forceinline__ uint32_t get_bits(const uint32_t *__restrict__ rowp, uint32_t b, uint32_t LB, uint32_t wpr)
{
    const uint32_t w = b >> 5, s = b & 31u;
    const uint32_t lo = rowp[w], hi = (w + 1u < wpr) ? rowp[w + 1u] : 0u;
    uint32_t v = __funnelshift_r(lo, hi, s);
    const uint32_t valid = LB - b;                          // bits left before the row wraps
    if (valid < 32u) v = (v & ((1u << valid) - 1u)) | (rowp[0] << valid);
    return v;
}

// Write nbits (> 0) bits to the row at bit position d0 (d0 + nbits <= LB, no wrap inside); fetch(i) returns 32 source bits
// starting at source bit i.
template <class Fetch>
__device__ __forceinline__ void put_range(uint32_t *rowp, uint32_t d0, uint32_t nbits, Fetch fetch)
{
    const uint32_t d1 = d0 + nbits;
    for (uint32_t j = d0 >> 5; j <= (d1 - 1u) >> 5; ++j) {
        const uint32_t lo = max(d0, j << 5), hi = min(d1, (j << 5) + 32u);       // destination bits [lo, hi) of word j
        const uint32_t n = hi - lo, sh = lo & 31u;
        const uint32_t mask = (n == 32u ? 0xFFFFFFFFu : ((1u << n) - 1u)) << sh;
        const uint32_t val = (fetch(lo - d0) << sh) & mask;
        if (mask == 0xFFFFFFFFu) rowp[j] = val;
        else { atomicAnd(rowp + j, ~mask); atomicOr(rowp + j, val); }
    }
}

template <int FB>
__global__ void __launch_bounds__(32) gthread_dt_kernel(Params p, uint32_t u, uint32_t colour, uint32_t nrows_win)
{
    using G = TGeom<6, FB>;                                  // window row pitch and field geometry of the S = 64 engine
    using At = Attempt<6, FB, 1>;                            // one lane per tile: 32 tiles per warp, whole-word store
    constexpr uint32_t PW = G::PW, NT = 32;
    extern __shared__ __align__(16) uint32_t smem[];
    const uint32_t lane = threadIdx.x;
    const uint32_t L = p.L, T = p.T, half = T >> 1, ntile = half * half;
    const uint32_t total = p.R * ntile;
    const uint32_t LB = L * FB, wpr = (LB + 31u) / 32u;
    uint32_t idx = blockIdx.x * NT + lane;
    const bool live = idx < total;
    if (!live) idx = total - 1u;                             // idle lanes shadow the last tile, write nothing
    const uint32_t rl = idx / ntile, n = idx - rl * ntile;
    const uint32_t I = 2u * (n % half) + (colour & 1u), J = 2u * (n / half) + (colour >> 1);
    const uint32_t rg = p.first_real + rl;
    (void)nrows_win;

    // D:2b: origin of sub-sweep u from the word stream of tile id 0xFFFFFFFF; tile edges floor(i L / T)
    uint32_t ox, oy;
    {
        WordStream os(p, 0xFFFFFFFFu, u, rg);
        const uint32_t thrL = pow32_mod(L);
        ox = os.draw(L, thrL);
        oy = os.draw(L, thrL);
    }
    const uint32_t bx = tile_edge(I, L, T), by = tile_edge(J, L, T);
    const uint32_t w = tile_edge(I + 1u, L, T) - bx, hgt = tile_edge(J + 1u, L, T) - by;
    const uint32_t x0 = (ox + bx) % L, y0 = (oy + by) % L;
    uint32_t *pk = p.pk + (size_t)rl * L * wpr;
    uint32_t *my = smem + lane;                              // word j of this lane's window: my[j * 32]
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(my);

    // ---- a3: window rows y0-1 .. y0+hgt; window column X <-> lattice column x0 - 1 + X (periodic) ---------------
    {
        const uint32_t xs = x0 ? x0 - 1u : L - 1u;
        const uint32_t b0 = xs * FB;
        for (uint32_t yr = 0; yr < hgt + 2u; ++yr) {
            uint32_t y = y0 + L - 1u + yr;
            y -= (y >= 2u * L) ? 2u * L : (y >= L ? L : 0u);
            const uint32_t *rowp = pk + (size_t)y * wpr;
#pragma unroll
            for (uint32_t k = 0; k < PW; ++k) {
                uint32_t b = b0 + 32u * k;
                if (b >= LB) b -= LB;
                my[(yr * PW + k) * NT] = get_bits(rowp, b, LB, wpr);
            }
        }
    }
    __syncwarp();

    // ---- a1 + a4: the tile's attempts in order (D:2b step 5) ----------------------------------------------------------
    uint32_t nacc = 0;
    {
        const uint32_t ns = w * hgt, thr = pow32_mod(ns);
        const uint64_t k = u & (p.K - 1u);
        const uint32_t A = (uint32_t)(((k + 1) * (uint64_t)ns) / p.K - (k * (uint64_t)ns) / p.K);
        const uint32_t N = p.N;
        const uint32_t inv_w = 0xFFFFFFFFu / w;              // s / w = mulhi(s, inv_w) or one more (s < 2^13)
        WordStream ws(p, J * T + I, u, rg);
        for (uint32_t a = 0; a < A; ++a) {
            const uint32_t s = ws.draw(ns, thr);
            uint32_t dy = __umulhi(s, inv_w);
            uint32_t dx = s - dy * w;
            if (dx >= w) { dx -= w; ++dy; }
            At at;
            const uint32_t bl = dx * FB, bc = bl + FB;       // window columns dx (left neighbour) and dx + 1 (site)
            const uint32_t row = base + (dy + 1u) * At::ROWB;
            at.a0 = row + (bl >> 5) * At::WSB;
            at.ac = row + (bc >> 5) * At::WSB;
            at.sl = bl & 31u;
            at.sc = bc & 31u;
            at.load();
            uint32_t nw;
            const bool ok = at.decide(N, nw);
            if (ok) at.store(nw);
            nacc += ok ? 1u : 0u;
        }
    }
    __syncwarp();

    // ---- a5: the w x hgt interior back into the packed lattice ------------------------------------------------------------
    if (live) {
        const uint32_t d0 = x0 * FB, nb = w * FB;
        for (uint32_t Y = 1; Y <= hgt; ++Y) {
            uint32_t y = y0 + Y - 1u;
            y -= y >= L ? L : 0u;
            uint32_t *rowp = pk + (size_t)y * wpr;
            // 32 bits of this window row starting at interior bit i (window bit FB + i)
            auto fetch_from = [&](uint32_t off) {
                return [=](uint32_t i) -> uint32_t {
                    const uint32_t b = FB + off + i, q = b >> 5;
                    const uint32_t lo = my[(Y * PW + q) * NT];
                    const uint32_t hi = (q + 1u < PW) ? my[(Y * PW + q + 1u) * NT] : 0u;
                    return __funnelshift_r(lo, hi, b & 31u);
                };
            };
            if (d0 + nb <= LB) put_range(rowp, d0, nb, fetch_from(0u));
            else {                                           // the tile row wraps around the end of the lattice row
                const uint32_t first = LB - d0;
                put_range(rowp, d0, first, fetch_from(0u));
                put_range(rowp, 0u, nb - first, fetch_from(first));
            }
        }
        if (nacc) atomicAdd(p.accepted + rl, (unsigned long long)nacc);
    }
}

// =============================================================================================
// Host side
// =============================================================================================
// General L, DT mode with S = 64, N <= 7, and both tile sizes within the window pitch of the S = 64 engine.
bool gthread_ok(uint32_t L, uint32_t N, uint32_t S, uint32_t K)
{
    if (S != 64 || N > 7 || 2 * S > L || (L & (L - 1)) == 0) return false;
    if ((S * S) % K || S * S / K < 32) return false;
    const uint32_t T = 2 * (L / (2 * S));
    return (L + T - 1) / T <= 66;
}

static uint32_t gthread_rows(const Params &p) { return (p.L + p.T - 1) / p.T + 2; }

size_t gthread_smem(const Params &p)
{
    const uint32_t pw = p.FB == 2 ? TGeom<6, 2>::PW : TGeom<6, 4>::PW;
    return (size_t)32 * pw * gthread_rows(p) * 4;
}

uint32_t gthread_blocks(const Params &p)
{
    const uint32_t half = p.T >> 1;
    return (uint32_t)(((uint64_t)p.R * half * half + 31) / 32);
}

cudaError_t gthread_configure(const Params &p)
{
    const int sm = (int)gthread_smem(p);
    return p.FB == 2 ? cudaFuncSetAttribute(gthread_dt_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm)
                     : cudaFuncSetAttribute(gthread_dt_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
}

cudaError_t gthread_launch(const Params &p, uint32_t u, uint32_t colour, cudaStream_t st)
{
    const size_t sm = gthread_smem(p);
    if (p.FB == 2) gthread_dt_kernel<2><<<gthread_blocks(p), 32, sm, st>>>(p, u, colour, gthread_rows(p));
    else gthread_dt_kernel<4><<<gthread_blocks(p), 32, sm, st>>>(p, u, colour, gthread_rows(p));
    return cudaGetLastError();
}

}  // namespace rsos
