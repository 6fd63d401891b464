// rsos_thread.cu -- the LANE-PER-TILE update engine of the DT schedule (sm_100a).
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// One colour pass of one sub-sweep (D:2 steps 4-6; RSOS rule P:61-63 Eq. 6; double tiling with a
// moving origin P:77; independent realizations P:75).  Every THREAD owns one active tile and runs
// its S*S/K attempts strictly in order, so the result is the sequential one by construction --
// no speculation, no votes.  What makes that fast (D:4, D:5):
//   * a site is FB bits, its height mod 2^FB (FB = 2 for N = 1, FB = 4 for N <= 7): under Eq. (6)
//     nearest-neighbour differences lie in [-N, N] and are recoverable mod 2^FB.  The working
//     lattice in HBM is packed the same way (rsos_pack.cu), so a tile window is (S+2) rows of
//     PW + 1 words instead of 4 bytes per site, and the int32 heights are rebuilt only on demand;
//   * the window of a lane is stored word-interleaved, word w of lane l at smem[w * 32 + l]: a
//     lane only ever touches bank l, so every shared-memory access of the attempt loop is
//     conflict-free (one wavefront per warp instruction);
//   * window column 0 is the left halo (the packed row is funnel-shifted while staging), so the
//     attempt loop has no per-tile alignment term.
#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace rsos {

template <int LGS, int FB>
struct TGeom {
    static constexpr uint32_t S = 1u << LGS;
    static constexpr uint32_t M = (1u << FB) - 1u;                 // field mask
    static constexpr uint32_t SPW = 32u / FB;                      // sites per word
    static constexpr uint32_t LGSPW = FB == 2 ? 4 : 3;
    static constexpr uint32_t WIN = S + 2;                         // window columns: halo, tile, halo
    static constexpr uint32_t PW = (WIN * FB + 31) / 32;           // words per window row
    static constexpr uint32_t ROWS = S + 2;
    static constexpr uint32_t WORDS = PW * ROWS;                   // words per lane
    static constexpr uint32_t ROWB = PW * 128;                     // byte stride of a row (interleaved)
    static constexpr uint32_t TBITS = S * FB;                      // bits of one tile row
    static constexpr uint32_t NTW = (TBITS + 31) / 32;             // words of one tile row
};

// One attempt at tile site (dx, dy) of this lane's tile; `base` = this lane's byte address of word
// 0 in shared memory.  Returns 1 if the deposit was accepted (D:2 step 6; D:3 (i)).
template <int LGS, int FB>
__device__ __forceinline__ uint32_t thread_attempt(uint32_t base, uint32_t dx, uint32_t dy, uint32_t N)
{
    using G = TGeom<LGS, FB>;
    constexpr uint32_t M = G::M;
    const uint32_t bl = dx * FB;                          // bit of the left neighbour (window column dx)
    const uint32_t bc = bl + FB;                          // bit of the site itself (window column dx + 1)
    const uint32_t row = base + (dy + 1u) * G::ROWB;
    const uint32_t a0 = row + (bl >> 5) * 128u;           // word holding the left neighbour
    const uint32_t ac = row + (bc >> 5) * 128u;           // word holding the site (and U/D columns)
    uint32_t w0, w1, wu, wd;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(w0) : "r"(a0));
    asm volatile("ld.shared.u32 %0, [%1+128];" : "=r"(w1) : "r"(a0));
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(wu) : "r"(ac - G::ROWB));
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(wd) : "r"(ac + G::ROWB));
    const uint32_t sc = bc & 31u;
    const uint32_t t3 = __funnelshift_r(w0, w1, bl & 31u);        // fields: L, C, R (garbage above)
    const uint32_t c = t3 >> FB;                                  // C in the low FB bits
    // Under Eq. (6) the deposit is rejected iff some neighbour sits at h - N, i.e. (C - nb) mod 2^FB == N
    // (D:3 (i)).  Branch-free: four independent subtract / test pairs.
    const uint32_t okL = ((c - t3) ^ N) & M;
    const uint32_t okR = ((c - (t3 >> (2 * FB))) ^ N) & M;
    const uint32_t okU = ((c - (wu >> sc)) ^ N) & M;
    const uint32_t okD = ((c - (wd >> sc)) ^ N) & M;
    const bool ok = (okL != 0u) & (okR != 0u) & (okU != 0u) & (okD != 0u);
    const uint32_t own = (bc >> 5) == (bl >> 5) ? w0 : w1;
    const uint32_t nw = own ^ (((c ^ (c + 1u)) & M) << sc);       // field + 1 mod 2^FB
    asm volatile("{ .reg .pred p; setp.ne.u32 p, %2, 0; @p st.shared.u32 [%0], %1; }"
                 :: "r"(ac), "r"(nw), "r"((uint32_t)ok) : "memory");
    return ok ? 1u : 0u;
}

// Block b runs tile set b: 32 active tiles, one per lane.
template <int LGS, int FB>
__global__ void __launch_bounds__(32) thread_dt_kernel(Params p, uint32_t u, uint32_t colour)
{
    using G = TGeom<LGS, FB>;
    constexpr uint32_t S = G::S, PW = G::PW, NTW = G::NTW;
    extern __shared__ __align__(16) uint32_t smem[];
    const uint32_t lane = threadIdx.x;
    const uint32_t L = p.L, Lm = L - 1;
    const uint32_t T = L >> LGS, half = T >> 1, ntile = half * half;
    const uint32_t total = p.R * ntile;
    uint32_t idx = blockIdx.x * 32u + lane;
    const bool live = idx < total;
    if (!live) idx = total - 1u;                         // idle lanes shadow the last tile, write nothing
    const uint32_t rl = idx / ntile, n = idx - rl * ntile;
    const uint32_t ti = n % half, tj = n / half;
    const uint32_t I = 2 * ti + (colour & 1u), J = 2 * tj + (colour >> 1);
    const uint32_t rg = p.first_real + rl;
    uint32_t ox, oy;
    draw_origin(p, u, rg, ox, oy);
    const uint32_t x0 = (ox + I * S) & Lm, y0 = (oy + J * S) & Lm;
    const uint32_t wpr = L >> G::LGSPW, wm = wpr - 1u;    // packed words per lattice row
    uint32_t *pk = p.pk + (size_t)rl * L * wpr;
    uint32_t *my = smem + lane;                           // word w of this lane: my[w * 32]
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(my);

    // ---- a3: stage rows y0-1 .. y0+S; window column X <-> lattice column x0 - 1 + X ------------
    {
        const uint32_t gxs = (x0 - 1u) & Lm;
        const uint32_t ws = gxs >> G::LGSPW, o = (gxs & (G::SPW - 1u)) * FB;
#pragma unroll 2
        for (uint32_t yr = 0; yr < G::ROWS; ++yr) {
            const uint32_t *rowp = pk + (size_t)((y0 - 1u + yr) & Lm) * wpr;
            uint32_t g[PW + 1];
#pragma unroll
            for (uint32_t k = 0; k <= PW; ++k) g[k] = rowp[(ws + k) & wm];
#pragma unroll
            for (uint32_t k = 0; k < PW; ++k) my[(yr * PW + k) * 32u] = __funnelshift_r(g[k], g[k + 1], o);
        }
    }
    __syncwarp();

    // ---- a1 + a4: A attempts in order; call q serves attempts 8q .. 8q+7 (16-bit slots) -------
    const uint32_t A = (S * S) / p.K;
    const uint32_t tile_id = J * T + I;
    const uint32_t N = p.N;
    uint32_t nacc = 0;
#pragma unroll 1
    for (uint32_t q = 0; q < A / 8u; ++q) {
        const uint4 o = philox4x32_10(q, tile_id, u, rg, p.k0, p.k1);
        const uint32_t ow[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
        for (uint32_t j = 0; j < 8; ++j) {
            const uint32_t v = (ow[j >> 1] >> (16u * (j & 1u))) & 0xFFFFu;
            nacc += thread_attempt<LGS, FB>(base, v & (S - 1u), (v >> LGS) & (S - 1u), N);
        }
    }
    __syncwarp();
    if (!live) return;

    // ---- a5: write back the S x S tile bits.  A tile row is TBITS bits starting at bit ob of
    // packed word wsb; whole words are stored, the (at most two) partial edge words are merged
    // with the lattice word.  No other tile of this pass touches those words: tiles of one colour
    // are S >= SPW sites apart (D:5).
    {
        const uint32_t wsb = x0 >> G::LGSPW, ob = (x0 & (G::SPW - 1u)) * FB;
#pragma unroll 1
        for (uint32_t Y = 1; Y <= S; ++Y) {
            uint32_t *rowp = pk + (size_t)((y0 - 1u + Y) & Lm) * wpr;
            uint32_t w[PW + 1];
#pragma unroll
            for (uint32_t k = 0; k < PW; ++k) w[k] = my[(Y * PW + k) * 32u];
            w[PW] = 0u;
            uint32_t tb[NTW + 2], tm[NTW + 2];             // tile bits / valid mask, padded with a zero word each side
            tb[0] = 0u; tm[0] = 0u; tb[NTW + 1] = 0u; tm[NTW + 1] = 0u;
#pragma unroll
            for (uint32_t k = 0; k < NTW; ++k) {
                const uint32_t full = (k + 1u) * 32u <= G::TBITS;
                const uint32_t mk = full ? 0xFFFFFFFFu : ((1u << (G::TBITS & 31u)) - 1u);
                tb[k + 1] = __funnelshift_r(w[k], w[k + 1], FB) & mk;   // drop the left halo column
                tm[k + 1] = mk;
            }
#pragma unroll
            for (uint32_t k = 0; k <= NTW; ++k) {
                const uint32_t gk = __funnelshift_l(tb[k], tb[k + 1], ob);
                const uint32_t mk = __funnelshift_l(tm[k], tm[k + 1], ob);
                uint32_t *dst = rowp + ((wsb + k) & wm);
                if (mk == 0xFFFFFFFFu) *dst = gk;
                else if (mk != 0u) *dst = (*dst & ~mk) | gk;
            }
        }
    }
    if (nacc) atomicAdd(p.accepted + rl, (unsigned long long)nacc);
}

// =============================================================================================
// Host-side launchers
// =============================================================================================
template <int LGS, int FB>
static cudaError_t thread_dt_t(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st, int what,
                               size_t *out)
{
    const size_t sm = (size_t)32 * TGeom<LGS, FB>::WORDS * 4;
    if (what == 0) { *out = sm; return cudaSuccess; }
    if (what == 1)
        return cudaFuncSetAttribute(thread_dt_kernel<LGS, FB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    thread_dt_kernel<LGS, FB><<<blocks, 32, sm, st>>>(p, u, colour);
    return cudaGetLastError();
}

static cudaError_t thread_dispatch(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st,
                                   int what, size_t *out)
{
    const bool two = p.FB == 2;
    switch (p.lgS) {
        case 3: return thread_dt_t<3, 4>(p, u, colour, blocks, st, what, out);      // S = 8 < 16 sites per 2-bit word
        case 4: return two ? thread_dt_t<4, 2>(p, u, colour, blocks, st, what, out)
                           : thread_dt_t<4, 4>(p, u, colour, blocks, st, what, out);
        case 5: return two ? thread_dt_t<5, 2>(p, u, colour, blocks, st, what, out)
                           : thread_dt_t<5, 4>(p, u, colour, blocks, st, what, out);
        case 6: return two ? thread_dt_t<6, 2>(p, u, colour, blocks, st, what, out)
                           : thread_dt_t<6, 4>(p, u, colour, blocks, st, what, out);
        default: return cudaErrorInvalidValue;
    }
}

// Field width of the packed lattice (D:5): 2 bits when N = 1 and a tile is at least one 2-bit
// word wide (so that tiles of one colour never share a packed word), else 4 bits (N <= 7).
uint32_t thread_dt_field_bits(uint32_t N, uint32_t S) { return (N <= 1u && S >= 16u) ? 2u : 4u; }

size_t thread_dt_smem(const Params &p)
{
    size_t sm = 0;
    thread_dispatch(p, 0, 0, 0, nullptr, 0, &sm);
    return sm;
}

cudaError_t thread_dt_configure(const Params &p) { return thread_dispatch(p, 0, 0, 0, nullptr, 1, nullptr); }

uint32_t thread_dt_blocks(const Params &p)
{
    const uint32_t T = p.L >> p.lgS, half = T >> 1;
    const uint64_t tiles = (uint64_t)p.R * half * half;
    return (uint32_t)((tiles + 31) / 32);
}

cudaError_t thread_dt_launch(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st)
{
    return thread_dispatch(p, u, colour, blocks, st, 2, nullptr);
}

}  // namespace rsos
