// rsos_fine.cu -- the FINE engine: DT schedule with small tiles ("cells") on lattices that live on chip (sm_100a).
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// SURVEY 8(f) NEXT-1 / P:83: for its steady-state runs (L = 64 ... 512) the paper used "domain sizes of 8 x 8
// lattice sites" as the finest sequential unit, and checked 16 x 16.  That is the schedule DT(c, K) of D:2
// with c = 8 or 16: (L / 2c)^2 cells per colour pass, c*c/K attempts each.  Per cell the work is tiny (64
// attempts), so what matters is never to leave the chip: a thread block keeps the whole lattice of one or more
// realizations in shared memory for every colour pass, sub-sweep and MCS of an rsos_advance call, one THREAD owns
// one cell of the current colour and runs its attempts in order straight on the resident lattice, and a block
// barrier separates the colour passes (cells of one colour are c sites apart, an attempt reads at distance <= 1
// and writes inside its cell: no two threads of a pass touch the same site).  No windows, no speculation,
// no votes.  The result is the oracle's DT(c, K), bit for bit; the W^2 bias of such small sequential units against
// serial dynamics (-3.6 % at c = 8, -1.6 % at c = 16) is the schedule's, and is measured in D:12.
//
// On-chip format: 4 bits per site (two sites per byte, site x in nibble x & 1 of byte x >> 1), holding the height
// mod 2^FB (FB = 2 or 4: the field width of the packed HBM lattice, D:5).  Active cells are >= 8 sites apart, so
// two threads never write the same byte.  L = 512 is 128 KiB, the largest lattice one block holds.
#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace rsos {

struct FineShape {
    uint32_t cpp;          // cells per colour pass of one realization = (L / 2c)^2
    uint32_t rpb;          // realizations per block
    uint32_t lat_words;    // 32-bit words of one on-chip lattice = L * L / 8
};

__device__ __forceinline__ uint32_t fine_lds_u8(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void fine_sts_u8(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u8 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// 8 two-bit fields (16 bits) -> 8 nibbles, and back.
__device__ __forceinline__ uint32_t spread8(uint32_t x)
{
    x = (x | (x << 8)) & 0x00FF00FFu;
    x = (x | (x << 4)) & 0x0F0F0F0Fu;
    return (x | (x << 2)) & 0x33333333u;
}
__device__ __forceinline__ uint32_t gather8(uint32_t x)
{
    x &= 0x33333333u;
    x = (x | (x >> 2)) & 0x0F0F0F0Fu;
    x = (x | (x >> 4)) & 0x00FF00FFu;
    return (x | (x >> 8)) & 0xFFFFu;
}

// Poisson variant DTP(c) (D:2c): attempt count of a cell in one sub-sweep from the 32-bit word w by inversion,
// n = #{k : w >= floor(2^32 P(X <= k))}, X ~ Poisson(4), k = 0 .. 22.
__constant__ uint32_t FINE_POISSON4[23] = {
    78665070u, 393325350u, 1022645910u, 1861739990u, 2700834071u, 3372109335u, 3819626178u, 4075350088u,
    4203212043u, 4260039579u, 4282770593u, 4291036416u, 4293791691u, 4294639467u, 4294881689u, 4294946282u,
    4294962430u, 4294966230u, 4294967074u, 4294967252u, 4294967287u, 4294967294u, 4294967295u};

__device__ __forceinline__ uint32_t poisson4_count(uint32_t w)
{
    uint32_t n = 0;
#pragma unroll
    for (int k = 0; k < 23; ++k) n += w >= FINE_POISSON4[k] ? 1u : 0u;
    return n;
}

template <int LGC, int FB, bool POISSON>
__global__ void __launch_bounds__(1024) fine_dt_kernel(Params p, uint32_t t0, uint32_t mcs, FineShape sh)
{
    constexpr uint32_t C = 1u << LGC, M = (1u << FB) - 1u;
    extern __shared__ __align__(16) uint32_t smem[];
    const uint32_t tid = threadIdx.x;
    const uint32_t L = p.L, Lm = L - 1u, lgL = p.lgL;
    const uint32_t T = L >> LGC, half = T >> 1;
    const uint32_t rs = tid / sh.cpp, n = tid - rs * sh.cpp;             // realization slot of the block, cell of the pass
    const uint32_t rl = blockIdx.x * sh.rpb + rs;
    const bool live = rs < sh.rpb && rl < p.R;
    const uint32_t rg = p.first_real + rl;
    const uint32_t nreal = min(sh.rpb, p.R - blockIdx.x * sh.rpb);        // realizations this block really holds

    // ---- load: packed HBM lattice (FB bits per site) -> 4 bits per site ------------------------------------------
    {
        const uint32_t pkw = sh.lat_words * FB / 4u;                     // packed words per realization
        const uint32_t *src = p.pk + (size_t)blockIdx.x * sh.rpb * pkw;
        for (uint32_t i = tid; i < nreal * pkw; i += blockDim.x) {
            const uint32_t v = src[i];
            if (FB == 4) smem[i] = v;
            else { smem[2u * i] = spread8(v & 0xFFFFu); smem[2u * i + 1u] = spread8(v >> 16); }
        }
    }
    __syncthreads();

    const uint32_t latb = (uint32_t)__cvta_generic_to_shared(smem + (live ? rs : 0u) * sh.lat_words);
    const uint32_t A = (C * C) / p.K, N = p.N;
    const uint32_t a_ = n % half, b_ = n / half;
    // A launch covers up to 2^36 attempts (rsos_api.cu) and on a small lattice with few realizations a thread owns a large
    // share of them: the count of one sub-sweep (at most a few hundred) is kept in 32 bits and folded into 64 after it.
    uint32_t nacc = 0;
    unsigned long long nacc_total = 0;

    for (uint32_t m = 0; m < mcs; ++m)
    for (uint32_t k = 0; k < p.K; ++k) {
        nacc_total += nacc;
        nacc = 0;
        const uint32_t u = (t0 + m) * p.K + k;
        uint32_t ox = 0, oy = 0;
        if (live) draw_origin(p, u, rg, ox, oy);
#pragma unroll 1
        for (uint32_t colour = 0; colour < 4; ++colour) {
            if (live) {
                const uint32_t I = 2u * a_ + (colour & 1u), J = 2u * b_ + (colour >> 1);
                const uint32_t x0 = (ox + I * C) & Lm, y0 = (oy + J * C) & Lm;
                const uint32_t tile_id = J * T + I;
                // one attempt with the 16-bit slot v (D:2 step 6); returns 1 if accepted
                auto attempt = [&](uint32_t v) -> uint32_t {
                    const uint32_t x = (x0 + (v & (C - 1u))) & Lm, y = (y0 + ((v >> LGC) & (C - 1u))) & Lm;
                    const uint32_t rowb = latb + (y << (lgL - 1u));
                    const uint32_t aC = rowb + (x >> 1);
                    const uint32_t bC = fine_lds_u8(aC);
                    const uint32_t bL = fine_lds_u8(rowb + (((x - 1u) & Lm) >> 1));
                    const uint32_t bR = fine_lds_u8(rowb + (((x + 1u) & Lm) >> 1));
                    const uint32_t bU = fine_lds_u8(latb + (((y - 1u) & Lm) << (lgL - 1u)) + (x >> 1));
                    const uint32_t bD = fine_lds_u8(latb + (((y + 1u) & Lm) << (lgL - 1u)) + (x >> 1));
                    const uint32_t s = (x & 1u) * 4u, sn = 4u - s;       // my nibble; x - 1 and x + 1 sit in the other one
                    const uint32_t c = bC >> s;
                    const uint32_t tq = (c - N) & M;                      // Eq. (6) under |dh| <= N: blocked iff a neighbour sits at h - N
                    const bool ok = (((bL >> sn) & M) != tq) & (((bR >> sn) & M) != tq) & (((bU >> s) & M) != tq) &
                                    (((bD >> s) & M) != tq);
                    if (ok) fine_sts_u8(aC, (bC & ~(15u << s)) | (((c + 1u) & M) << s));
                    return ok ? 1u : 0u;
                };
                if (POISSON) {
                    // D:2c: n ~ Poisson(4) attempts from the first word of Philox call 0xFFFFFFFF of this cell
                    const uint32_t cnt = poisson4_count(philox4x32_10(0xFFFFFFFFu, tile_id, u, rg, p.k0, p.k1).x);
                    uint4 o = make_uint4(0, 0, 0, 0);
#pragma unroll 1
                    for (uint32_t a = 0; a < cnt; ++a) {
                        const uint32_t w = a & 7u;
                        if (w == 0u) o = philox4x32_10(a >> 3, tile_id, u, rg, p.k0, p.k1);
                        const uint32_t word = (w >> 1) == 0u ? o.x : (w >> 1) == 1u ? o.y : (w >> 1) == 2u ? o.z : o.w;
                        nacc += attempt((w & 1u) ? word >> 16 : word);
                    }
                } else {
#pragma unroll 1
                    for (uint32_t q = 0; q < A / 8u; ++q) {
                        const uint4 o = philox4x32_10(q, tile_id, u, rg, p.k0, p.k1);
                        const uint32_t ow[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
                        for (uint32_t w = 0; w < 8; ++w)                 // slot w of call q
                            nacc += attempt((w & 1u) ? ow[w >> 1] >> 16 : ow[w >> 1]);
                    }
                }
            }
            __syncthreads();                                             // the next colour reads what this one wrote
        }
    }

    // ---- store: 4 bits per site -> packed lattice; accepted counts ------------------------------------------------
    {
        const uint32_t pkw = sh.lat_words * FB / 4u;
        uint32_t *dst = p.pk + (size_t)blockIdx.x * sh.rpb * pkw;
        for (uint32_t i = tid; i < nreal * pkw; i += blockDim.x) {
            if (FB == 4) dst[i] = smem[i];
            else dst[i] = gather8(smem[2u * i]) | (gather8(smem[2u * i + 1u]) << 16);
        }
    }
    nacc_total += nacc;
    if (live && nacc_total) atomicAdd(p.accepted + rl, nacc_total);
}

// =============================================================================================
// Host side
// =============================================================================================
constexpr size_t FINE_SMEM_BUDGET = 128u * 1024u;       // lattice bytes per block (L = 512 at 4 bits per site)

static bool fine_shape(uint32_t L, uint32_t S, uint32_t R, uint32_t sm_count, FineShape *sh)
{
    const uint32_t half = L / S / 2;
    sh->cpp = half * half;
    sh->lat_words = L * L / 8;
    if (sh->cpp > 1024u || (size_t)sh->lat_words * 4 > FINE_SMEM_BUDGET) return false;
    // 256 threads per block when that still gives every SM a block, else 64 (one thread per cell is all the
    // parallelism a pass has: R (L / 2c)^2 threads); one realization per block when a pass has that many cells
    const uint64_t total = (uint64_t)R * sh->cpp;
    const uint32_t tpb = total >= (uint64_t)(sm_count ? sm_count : 1u) * 256u ? 256u : 64u;
    uint32_t rpb = tpb / sh->cpp;
    if (rpb > R) rpb = R;
    sh->rpb = rpb ? rpb : 1u;
    return true;
}

// DT mode, cells of 8 or 16 sites, N <= 7, the 4-bit lattice of one realization within 128 KiB (L <= 512).
bool fine_ok(uint32_t L, uint32_t N, uint32_t S, uint32_t K, bool poisson)
{
    if ((S != 8 && S != 16) || N > 7 || 2 * S > L || L > 512) return false;
    if (poisson) return K == S * S / 4;
    return (S * S) % K == 0 && S * S / K >= 8 && (S * S / K) % 8 == 0;
}

template <int LGC, int FB, bool POISSON>
static cudaError_t fine_t(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st, int what, uint32_t *out)
{
    FineShape sh;
    if (!fine_shape(p.L, p.S, p.R, p.sm_count, &sh)) return cudaErrorInvalidValue;
    const size_t sm = (size_t)sh.rpb * sh.lat_words * 4;
    const uint32_t threads = (sh.rpb * sh.cpp + 31u) / 32u * 32u;
    const uint32_t blocks = (p.R + sh.rpb - 1) / sh.rpb;
    if (what == 0) { out[0] = (uint32_t)sm; out[1] = blocks; out[2] = threads; out[3] = sh.rpb; return cudaSuccess; }
    if (what == 1) return cudaFuncSetAttribute(fine_dt_kernel<LGC, FB, POISSON>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    fine_dt_kernel<LGC, FB, POISSON><<<blocks, threads, sm, st>>>(p, t0, mcs, sh);
    return cudaGetLastError();
}

static cudaError_t fine_dispatch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st, int what, uint32_t *out)
{
    if (p.poisson) {
        if (p.lgS == 3) return fine_t<3, 4, true>(p, t0, mcs, st, what, out);
        if (p.lgS == 4) return p.FB == 2 ? fine_t<4, 2, true>(p, t0, mcs, st, what, out) : fine_t<4, 4, true>(p, t0, mcs, st, what, out);
        return cudaErrorInvalidValue;
    }
    if (p.lgS == 3) return fine_t<3, 4, false>(p, t0, mcs, st, what, out);   // 8-site cells: 4-bit packed lattice (D:5)
    if (p.lgS == 4) return p.FB == 2 ? fine_t<4, 2, false>(p, t0, mcs, st, what, out) : fine_t<4, 4, false>(p, t0, mcs, st, what, out);
    return cudaErrorInvalidValue;
}

size_t fine_smem(const Params &p) { uint32_t o[4] = {0, 0, 0, 0}; fine_dispatch(p, 0, 0, nullptr, 0, o); return o[0]; }
uint32_t fine_blocks(const Params &p) { uint32_t o[4] = {0, 0, 0, 0}; fine_dispatch(p, 0, 0, nullptr, 0, o); return o[1]; }
cudaError_t fine_configure(const Params &p) { return fine_dispatch(p, 0, 0, nullptr, 1, nullptr); }
cudaError_t fine_launch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st) { return fine_dispatch(p, t0, mcs, st, 2, nullptr); }

}  // namespace rsos
