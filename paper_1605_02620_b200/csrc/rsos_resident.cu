// rsos_resident.cu -- the RESIDENT engine: DT schedule on lattices small enough to live on chip (sm_100a).
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// BASELINE.json north_star (3) / P:75: "a whole lattice lives on-chip for many sweeps".  When a
// colour pass of the DT schedule (D:2 steps 4-6) has only a few tiles per realization (L = 128
// ... 512 at S = 64: 1, 4, 16), launching one kernel per pass re-stages every tile from global memory
// 4K times per MCS and leaves the machine to launch latency.  Here one thread block owns one
// realization for ALL colour passes, sub-sweeps and MCS of an rsos_advance call:
//   * the packed lattice (FB = 2 or 4 bits per site, D:5, the same format as the THREAD engine's HBM
//     working state) is loaded once into shared memory, periodic, row-major;
//   * per pass every group of KL lanes copies its tile window (S + 2)^2 out of the resident lattice
//     into the window format of rsos_attempt.cuh (shared -> shared, column 0 = left halo), runs its
//     S*S/K attempts in order, and copies the S x S interior back; one block barrier per pass;
//   * KL = 8, 16 or 32 lanes work on one tile: in every step they take KL consecutive attempts on one
//     snapshot.  A lane whose site may interact with the site of a LOWER rank (equal, adjacent, or in
//     the same byte of packed sites) is "hazardous": it waits for the lower ranks and decides again.
//     The hazard test needs only the site codes, which are pure functions of the Philox counter, so
//     it is computed one step ahead, with three MATCH.ANY instructions on overlapping coarse cells
//     (see hazard_mask) -- exact sequential semantics, checked bit for bit against the oracle;
//   * the 16-bit Philox slots of a batch of 8 steps go through a small shared-memory table (one
//     128-bit store per lane and batch, one 16-bit load per lane and step).
#include "rsos_attempt.cuh"
#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace rsos {

// Lower-rank lanes of my group whose attempt may interact with mine.  Two sites interact if they are
// equal, nearest neighbours, or share a byte of the packed window row (byte stores).  Window column
// X = dx + 1 holds site dx; a byte holds SPB = 8 / FB consecutive columns.  Cover the window with
// three grids of cells SPB wide and 2 tall:  A = aligned,  B = shifted by SPB / 2 in x,  C = shifted
// by 1 in y.  Equal sites and sites in one byte share an A cell; horizontal neighbours share an A or
// a B cell (x and x + 1 are split by at most one of the two x-grids, and y-cells agree); vertical
// neighbours share an A or a C cell.  So  interact(i, j)  =>  same cell in A, B or C, and the union of
// three MATCH.ANY results is a conservative hazard mask (a false alarm costs a reload, never a wrong
// result).  The group index is part of the matched value, so groups never see each other.
template <int LGS, int FB>
__device__ __forceinline__ uint32_t hazard_mask(uint32_t v, uint32_t grp, uint32_t lower_in_group)
{
    constexpr uint32_t S = 1u << LGS;
    constexpr uint32_t XS = FB == 2 ? 2u : 1u;                         // lg(sites per byte)
    const uint32_t X = (v & (S - 1u)) + 1u, dy = (v >> LGS) & (S - 1u);
    const uint32_t ya = dy >> 1, yc = (dy + 1u) >> 1;                  // < 64 for S <= 64
    const uint32_t xa = X >> XS, xb = (X + (1u << (XS - 1u))) >> XS;   // < 64
    const uint32_t g = grp << 12;
    const uint32_t mA = __match_any_sync(0xFFFFFFFFu, g | (ya << 6) | xa);
    const uint32_t mB = __match_any_sync(0xFFFFFFFFu, g | (ya << 6) | xb);
    const uint32_t mC = __match_any_sync(0xFFFFFFFFu, g | (yc << 6) | xa);
    return (mA | mB | mC) & lower_in_group;
}

struct ResidentShape {
    uint32_t tpp;          // tiles per colour pass of one realization = (L / 2S)^2
    uint32_t rpb;          // realizations per block
    uint32_t threads;      // rpb * tpp * KL
};

// One block = rpb realizations.  Shared memory: [rpb lattices][per warp: NT windows][per warp: 2 slot tables].
template <int LGS, int FB, int KL>
__global__ void __launch_bounds__(KL * 16 < 32 ? 32 : KL * 16) resident_dt_kernel(Params p, uint32_t t0, uint32_t mcs, ResidentShape sh)
{
    using G = TGeom<LGS, FB>;
    using At = Attempt<LGS, FB, KL>;
    constexpr uint32_t S = G::S, PW = G::PW, NTW = G::NTW, NT = At::NT;
    constexpr uint32_t FULL = 0xFFFFFFFFu;
    extern __shared__ __align__(16) uint32_t smem[];
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t nwarps = blockDim.x >> 5;
    const uint32_t grp = lane / KL, rank = lane % KL;
    const uint32_t L = p.L, Lm = L - 1u;
    const uint32_t wpr = L >> G::LGSPW, wm = wpr - 1u;               // packed words per lattice row
    const uint32_t lat_words = L * wpr;
    const uint32_t T = L >> LGS, half = T >> 1;

    uint32_t *lat_all = smem;
    uint32_t *win = smem + sh.rpb * lat_words + warp * (NT * G::WORDS);
    uint32_t *tab = smem + sh.rpb * lat_words + nwarps * (NT * G::WORDS) + warp * 256u;   // 2 x 32 lanes x 4 words

    // which tile of which realization this group works on
    const uint32_t gt = warp * NT + grp;                             // group index in the block
    const uint32_t rb = gt / sh.tpp, n = gt - rb * sh.tpp;
    const uint32_t rl0 = blockIdx.x * sh.rpb;
    const uint32_t rl = rl0 + rb;
    const bool live = rl < p.R;
    const uint32_t ti = n % half, tj = n / half;
    const uint32_t rg = p.first_real + (live ? rl : p.R - 1u);
    uint32_t *lat = lat_all + rb * lat_words;

    // ---- load the packed lattices of this block (coalesced 128-bit) -------------------------------
    {
        const uint32_t nreal = min(sh.rpb, p.R - rl0);
        const uint4 *src = reinterpret_cast<const uint4 *>(p.pk + (size_t)rl0 * lat_words);
        uint4 *dst = reinterpret_cast<uint4 *>(lat_all);
        for (uint32_t i = tid; i < nreal * lat_words / 4u; i += blockDim.x) dst[i] = src[i];
    }
    __syncthreads();

    uint32_t *my = win + grp;                                         // word w of this group's window: my[w * NT]
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(my);
    const uint32_t tabb = (uint32_t)__cvta_generic_to_shared(tab);
    const uint32_t lower = ((1u << rank) - 1u) << (grp * KL);          // lower ranks of my group
    const uint32_t A = (S * S) / p.K;
    const uint32_t nbatch = A / (8u * KL);
    const uint32_t N = p.N;
    unsigned long long nacc = 0;

    for (uint32_t m = 0; m < mcs; ++m)
    for (uint32_t k = 0; k < p.K; ++k) {
        const uint32_t u = (t0 + m) * p.K + k;
        uint32_t ox, oy;
        draw_origin(p, u, rg, ox, oy);
#pragma unroll 1
        for (uint32_t colour = 0; colour < 4; ++colour) {
            const uint32_t I = 2 * ti + (colour & 1u), J = 2 * tj + (colour >> 1);
            const uint32_t x0 = (ox + I * S) & Lm, y0 = (oy + J * S) & Lm;
            const uint32_t tile_id = J * T + I;

            // ---- a3: window rows y0-1 .. y0+S out of the resident lattice; column X <-> x0 - 1 + X ----
            {
                const uint32_t gxs = (x0 - 1u) & Lm;
                const uint32_t ws = gxs >> G::LGSPW, o = (gxs & (G::SPW - 1u)) * FB;
#pragma unroll 1
                for (uint32_t yr = rank; yr < G::ROWS; yr += KL) {
                    const uint32_t *rowp = lat + ((y0 - 1u + yr) & Lm) * wpr;
                    uint32_t g[PW + 1];
#pragma unroll
                    for (uint32_t q = 0; q <= PW; ++q) g[q] = rowp[(ws + q) & wm];
#pragma unroll
                    for (uint32_t q = 0; q < PW; ++q) my[(yr * PW + q) * NT] = __funnelshift_r(g[q], g[q + 1], o);
                }
            }
            // first batch of slots: rank r computes Philox call r of the tile (D:2 step 6)
            {
                const uint4 c = philox4x32_10(rank, tile_id, u, rg, p.k0, p.k1);
                asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(tabb + lane * 16u), "r"(c.x), "r"(c.y), "r"(c.z), "r"(c.w) : "memory");
            }
            __syncwarp();

            // ---- a1 + a4: A attempts in order, KL per step; attempt e of a batch reads the 16-bit slot e
            // of the group's table (call e >> 3, slot e & 7) ------------------------------------------------
            auto slot = [&](uint32_t buf, uint32_t w) -> uint32_t {
                uint32_t v;
                asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(tabb + buf * 512u + grp * (KL * 16u) + (KL * w + rank) * 2u));
                return v;
            };
            At cur;
            uint32_t v0 = slot(0u, 0u);
            cur.prep(base, v0);
            uint32_t hm = hazard_mask<LGS, FB>(v0, grp, lower);
#pragma unroll 1
            for (uint32_t batch = 0; batch < nbatch; ++batch) {
                const uint32_t buf = batch & 1u;
                {   // slots of the next batch (unused after the last one)
                    const uint4 c = philox4x32_10((batch + 1u) * KL + rank, tile_id, u, rg, p.k0, p.k1);
                    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(tabb + (buf ^ 1u) * 512u + lane * 16u), "r"(c.x), "r"(c.y), "r"(c.z), "r"(c.w) : "memory");
                }
#pragma unroll
                for (uint32_t w = 0; w < 8; ++w) {
                    cur.load();
                    // next step's slot, addresses and hazard mask depend on nothing in the window
                    const uint32_t vn = w < 7u ? slot(buf, w + 1u) : slot(buf ^ 1u, 0u);
                    At nxt;
                    nxt.prep(base, vn);
                    const uint32_t hmn = hazard_mask<LGS, FB>(vn, grp, lower);
                    uint32_t nw;
                    bool ok = cur.decide(N, nw);
                    bool wait = hm != 0u;
                    if (ok & !wait) cur.store(nw);
                    __syncwarp();
                    uint32_t pend = __ballot_sync(FULL, wait);
                    while (pend) {
                        // ready: pending, and no lower rank I may interact with is still pending
                        const bool ready = wait & ((hm & pend) == 0u);
                        if (ready) {
                            cur.load();
                            ok = cur.decide(N, nw);
                            if (ok) cur.store(nw);
                            wait = false;
                        }
                        __syncwarp();
                        pend &= ~__ballot_sync(FULL, ready);
                    }
                    nacc += ok ? 1u : 0u;
                    cur = nxt;
                    hm = hmn;
                }
            }
            __syncwarp();

            // ---- a5: the S x S interior back into the resident lattice (plain read-modify-write of the two
            // partial edge words: no other tile of this pass touches them, tiles of a colour are 2S apart) ----
            {
                const uint32_t wsb = x0 >> G::LGSPW, ob = (x0 & (G::SPW - 1u)) * FB;
#pragma unroll 1
                for (uint32_t Y = 1u + rank; Y <= S; Y += KL) {
                    uint32_t *rowp = lat + ((y0 - 1u + Y) & Lm) * wpr;
                    uint32_t w[PW + 1];
#pragma unroll
                    for (uint32_t q = 0; q < PW; ++q) w[q] = my[(Y * PW + q) * NT];
                    w[PW] = 0u;
                    uint32_t tb[NTW + 2], tm[NTW + 2];
                    tb[0] = 0u; tm[0] = 0u; tb[NTW + 1] = 0u; tm[NTW + 1] = 0u;
#pragma unroll
                    for (uint32_t q = 0; q < NTW; ++q) {
                        const uint32_t full = (q + 1u) * 32u <= G::TBITS;
                        const uint32_t mk = full ? 0xFFFFFFFFu : ((1u << (G::TBITS & 31u)) - 1u);
                        tb[q + 1] = __funnelshift_r(w[q], w[q + 1], FB) & mk;      // drop the left halo column
                        tm[q + 1] = mk;
                    }
#pragma unroll
                    for (uint32_t q = 0; q <= NTW; ++q) {
                        const uint32_t gk = __funnelshift_l(tb[q], tb[q + 1], ob);
                        const uint32_t mk = __funnelshift_l(tm[q], tm[q + 1], ob);
                        uint32_t *dst = rowp + ((wsb + q) & wm);
                        if (mk == 0xFFFFFFFFu) *dst = gk;
                        else if (mk != 0u) *dst = (*dst & ~mk) | gk;
                    }
                }
            }
            __syncthreads();                                       // the next pass reads what this one wrote
        }
    }

    // ---- store the lattices, add the accepted counts ---------------------------------------------------
    {
        const uint32_t nreal = min(sh.rpb, p.R - rl0);
        uint4 *dst = reinterpret_cast<uint4 *>(p.pk + (size_t)rl0 * lat_words);
        const uint4 *src = reinterpret_cast<const uint4 *>(lat_all);
        for (uint32_t i = tid; i < nreal * lat_words / 4u; i += blockDim.x) dst[i] = src[i];
    }
    // group sum of nacc (KL lanes, contiguous), then one atomic per group
#pragma unroll
    for (uint32_t o = KL / 2; o; o >>= 1) nacc += __shfl_xor_sync(FULL, nacc, o);
    if (rank == 0 && live && nacc) atomicAdd(p.accepted + rl, nacc);
}

// =============================================================================================
// Host side
// =============================================================================================
static bool shape_of(const Params &p, uint32_t KL, ResidentShape *sh)
{
    const uint32_t half = (p.L >> p.lgS) >> 1;
    sh->tpp = half * half;
    const uint32_t per_real = sh->tpp * KL;                         // threads one realization needs
    if (sh->tpp > 16u) return false;                                // launch bounds of the kernel: 16 * KL threads
    sh->rpb = per_real >= 32u ? 1u : 32u / per_real;
    sh->threads = sh->rpb * per_real;
    return sh->threads % 32u == 0u;
}

template <int LGS, int FB>
static size_t smem_of(const Params &p, uint32_t KL, const ResidentShape &sh)
{
    const size_t lat_words = (size_t)p.L * (p.L * FB / 32);
    const size_t warps = sh.threads / 32, nt = 32 / KL;
    return (sh.rpb * lat_words + warps * nt * TGeom<LGS, FB>::WORDS + warps * 256) * 4;
}

// what: 0 = shared-memory bytes (*out), 1 = set the function attribute, 2 = launch
template <int LGS, int FB, int KL>
static cudaError_t resident_t(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st, int what, size_t *out)
{
    ResidentShape sh;
    if (!shape_of(p, KL, &sh)) return cudaErrorInvalidValue;
    const size_t sm = smem_of<LGS, FB>(p, KL, sh);
    if (what == 0) { *out = sm; return cudaSuccess; }
    if (what == 1)
        return cudaFuncSetAttribute(resident_dt_kernel<LGS, FB, KL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    const uint32_t blocks = (p.R + sh.rpb - 1) / sh.rpb;
    resident_dt_kernel<LGS, FB, KL><<<blocks, sh.threads, sm, st>>>(p, t0, mcs, sh);
    return cudaGetLastError();
}

template <int LGS, int FB>
static cudaError_t resident_k(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st, int what, size_t *out)
{
    switch (p.KL) {
        case 4: return resident_t<LGS, FB, 4>(p, t0, mcs, st, what, out);
        case 8: return resident_t<LGS, FB, 8>(p, t0, mcs, st, what, out);
        case 16: return resident_t<LGS, FB, 16>(p, t0, mcs, st, what, out);
        case 32: return resident_t<LGS, FB, 32>(p, t0, mcs, st, what, out);
        default: return cudaErrorInvalidValue;
    }
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

// Can the RESIDENT engine run (L, N, S, K) with KL lanes per tile within smem_limit bytes per block?
// Needs DT mode, 16 <= S <= 64, N <= 7, a batch of 8 * KL attempts dividing S*S/K, at most 1024
// threads per realization, and the packed lattice plus windows in shared memory.
bool resident_ok(uint32_t L, uint32_t N, uint32_t S, uint32_t K, uint32_t KL, size_t smem_limit)
{
    if (S < 16 || S > 64 || N > 7 || 2 * S > L) return false;
    if (KL != 4 && KL != 8 && KL != 16 && KL != 32) return false;
    const uint32_t A = S * S / K;
    if (A % (8 * KL)) return false;
    Params p{};
    p.L = L; p.lgS = S == 16 ? 4 : S == 32 ? 5 : 6; p.FB = thread_dt_field_bits(N, S); p.KL = KL;
    ResidentShape sh;
    if (!shape_of(p, KL, &sh)) return false;
    size_t sm = 0;
    if (resident_dispatch(p, 0, 0, nullptr, 0, &sm) != cudaSuccess) return false;
    return sm <= smem_limit;
}

size_t resident_smem(const Params &p)
{
    size_t sm = 0;
    resident_dispatch(p, 0, 0, nullptr, 0, &sm);
    return sm;
}

cudaError_t resident_configure(const Params &p) { return resident_dispatch(p, 0, 0, nullptr, 1, nullptr); }

uint32_t resident_blocks(const Params &p)
{
    ResidentShape sh;
    if (!shape_of(p, p.KL, &sh)) return 0;
    return (p.R + sh.rpb - 1) / sh.rpb;
}

// `mcs` whole MCS starting at sweep counter t0, all colour passes and sub-sweeps inside one launch.
cudaError_t resident_launch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st)
{
    return resident_dispatch(p, t0, mcs, st, 2, nullptr);
}

}  // namespace rsos
