// rsos_thread.cu -- the LANE-PER-TILE update engine of the DT schedule (sm_100a).
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// One colour pass of one sub-sweep (D:2 steps 4-6; RSOS rule P:61-63 Eq. 6; double tiling with a
// moving origin P:77; independent realizations P:75).  Every THREAD owns one active tile and runs
// its S*S/K attempts strictly in order, so the result is the sequential one by construction --
// no speculation, no votes.  What makes that fast (D:4):
//   * on chip a site is FB bits: its height mod 2^FB (FB = 2 for N = 1, FB = 4 for N <= 7; any
//     nearest-neighbour difference lies in [-N, N] under Eq. (6), so it is recoverable mod 2^FB);
//   * the (S+2)-row window of a lane is stored word-interleaved, word w of lane l at
//     smem[w * 32 + l]: a lane only ever touches bank l, so every shared-memory access of the
//     attempt loop is conflict-free (one wavefront per warp instruction);
//   * the window keeps the 4-aligned global columns [xa, xa + S + 8) unshifted, so staging is
//     int4 loads and write-back is int4 stores;
//   * int32 heights are rebuilt at write-back from ONE global value per tile (the window's
//     top-left corner) by difference chains: down column 0, then along every row.
#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace rsos {

template <int LGS, int FB>
struct TGeom {
    static constexpr uint32_t S = 1u << LGS;
    static constexpr uint32_t M = (1u << FB) - 1u;                 // field mask
    static constexpr uint32_t WIN = S + 8;                         // window columns (sites)
    static constexpr uint32_t NCH = WIN / 4;                       // int4 chunks per window row
    static constexpr uint32_t PW = (WIN * FB + 31) / 32;           // words per window row
    static constexpr uint32_t ROWS = S + 2;
    static constexpr uint32_t WORDS = PW * ROWS;                   // words per lane
    static constexpr uint32_t ROWB = PW * 128;                     // byte stride of a row (interleaved)
};

// low FB bits of four heights -> 4*FB bits, site k at bit k*FB
template <int FB>
__device__ __forceinline__ uint32_t pack4(const int4 q)
{
    constexpr uint32_t M = (1u << FB) - 1u;
    return ((uint32_t)q.x & M) | (((uint32_t)q.y & M) << FB) | (((uint32_t)q.z & M) << (2 * FB)) |
           (((uint32_t)q.w & M) << (3 * FB));
}

// sign-extended FB-bit field of d at bit position pos (compile-time)
template <int FB>
__device__ __forceinline__ int32_t sfield(uint32_t d, int pos)
{
    return ((int32_t)(d << (32 - FB - pos))) >> (32 - FB);
}

// One attempt at window site (X, Y) of this lane's tile; `base` = this lane's byte address of
// word 0 in shared memory.  Returns 1 if the deposit was accepted (D:2 step 6; D:3 (i)).
template <int LGS, int FB>
__device__ __forceinline__ uint32_t thread_attempt(uint32_t base, uint32_t dx, uint32_t dy, uint32_t offx,
                                                   uint32_t N)
{
    using G = TGeom<LGS, FB>;
    constexpr uint32_t M = G::M;
    const uint32_t X = dx + offx, Y = dy + 1u;
    const uint32_t bl = (X - 1u) * FB;                    // bit of the left neighbour in the row
    const uint32_t bc = bl + FB;                          // bit of the site itself
    const uint32_t row = base + Y * G::ROWB;
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

template <int LGS, int FB>
__global__ void __launch_bounds__(32) thread_dt_kernel(Params p, uint32_t u, uint32_t colour)
{
    using G = TGeom<LGS, FB>;
    constexpr uint32_t S = G::S, PW = G::PW, NCH = G::NCH;
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
    const uint32_t offx = ((x0 - 1u) & 3u) + 1u;          // window column of tile column 0 (1..4)
    const uint32_t xa = (x0 - offx) & Lm;                 // global column of window column 0 (multiple of 4)
    int32_t *h = p.h + (size_t)rl * L * L;
    uint32_t *my = smem + lane;                           // word w of this lane: my[w * 32]
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(my);

    // ---- a3: stage rows y0-1 .. y0+S, window columns 0 .. S+7, FB bits per site ---------------
#pragma unroll 1
    for (uint32_t yr = 0; yr < G::ROWS; ++yr) {
        const int32_t *grow = h + (size_t)((y0 - 1u + yr) & Lm) * L;
        uint32_t wbuf[PW];
#pragma unroll
        for (uint32_t k = 0; k < PW; ++k) wbuf[k] = 0u;
#pragma unroll
        for (uint32_t c = 0; c < NCH; ++c) {
            const int4 q = __ldg(reinterpret_cast<const int4 *>(grow + ((xa + 4u * c) & Lm)));
            const uint32_t bit = c * 4u * FB;
            wbuf[bit >> 5] |= pack4<FB>(q) << (bit & 31u);
        }
#pragma unroll
        for (uint32_t k = 0; k < PW; ++k) my[(yr * PW + k) * 32u] = wbuf[k];
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
            nacc += thread_attempt<LGS, FB>(base, v & (S - 1u), (v >> LGS) & (S - 1u), offx, N);
        }
    }
    __syncwarp();
    if (!live) return;

    // ---- a5: write back.  h(0, Y) by a chain down window column 0 from the corner value; then
    // along row Y:  h(X) = h(X-1) + sext(b(X) - b(X-1)).  Adjacent sites differ by <= N everywhere
    // (Eq. 6 holds on frozen and active sites alike), so FB bits recover every difference.
    int32_t hcol = h[(size_t)((y0 - 1u) & Lm) * L + xa];
    uint32_t bcol = my[0] & G::M;
#pragma unroll 1
    for (uint32_t Y = 1; Y <= S; ++Y) {
        uint32_t w[PW];
#pragma unroll
        for (uint32_t k = 0; k < PW; ++k) w[k] = my[(Y * PW + k) * 32u];
        const uint32_t b0 = w[0] & G::M;
        hcol += sfield<FB>(b0 - bcol, 0);
        bcol = b0;
        int32_t *grow = h + (size_t)((y0 - 1u + Y) & Lm) * L;
        int32_t cur = hcol;
#pragma unroll
        for (uint32_t c = 0; c < NCH - 1u; ++c) {          // the last chunk is never inside the tile
            int32_t out[4];
#pragma unroll
            for (uint32_t e = 0; e < 4; ++e) {
                const uint32_t Xs = 4u * c + e;
                const uint32_t bit = Xs * FB;
                const uint32_t wk = w[bit >> 5];
                uint32_t d;                                  // b(Xs) - b(Xs-1) in the low FB bits
                if (Xs == 0u) d = 0u;
                else if ((bit & 31u) == 0u) d = wk - (w[(bit >> 5) - 1u] >> (32 - FB));
                else d = (wk >> (bit & 31u)) - (wk >> ((bit & 31u) - FB));
                cur += sfield<FB>(d, 0);
                out[e] = cur;
            }
            const uint32_t gx = (xa + 4u * c) & Lm;
            const uint32_t Xlo = 4u * c;
            if (c != 0u && c != NCH - 2u) {                 // chunks 1 .. NCH-3 lie inside the tile for every offx
                *reinterpret_cast<int4 *>(grow + gx) = make_int4(out[0], out[1], out[2], out[3]);
            } else {
#pragma unroll
                for (uint32_t e = 0; e < 4; ++e)
                    if (Xlo + e >= offx && Xlo + e <= offx + S - 1u) grow[gx + e] = out[e];
            }
        }
    }
    if (nacc) atomicAdd(p.accepted + rl, (unsigned long long)nacc);
}

// =============================================================================================
// Host-side launchers
// =============================================================================================
template <int LGS, int FB>
static cudaError_t thread_dt_t(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, uint32_t pf_stride,
                               cudaStream_t st, int what, size_t *out)
{
    const size_t sm = (size_t)32 * TGeom<LGS, FB>::WORDS * 4;
    if (what == 0) { *out = sm; return cudaSuccess; }
    if (what == 1)
        return cudaFuncSetAttribute(thread_dt_kernel<LGS, FB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (what == 3) {                                      // resident blocks per SM
        int nb = 0;
        const cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, thread_dt_kernel<LGS, FB>, 32, sm);
        *out = (size_t)nb;
        return e;
    }
    (void)pf_stride;
    thread_dt_kernel<LGS, FB><<<blocks, 32, sm, st>>>(p, u, colour);
    return cudaGetLastError();
}

static cudaError_t thread_dispatch(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, uint32_t pf_stride,
                                   cudaStream_t st, int what, size_t *out)
{
    const bool two = p.N <= 1;
    switch (p.lgS) {
        case 3: return two ? thread_dt_t<3, 2>(p, u, colour, blocks, pf_stride, st, what, out)
                           : thread_dt_t<3, 4>(p, u, colour, blocks, pf_stride, st, what, out);
        case 4: return two ? thread_dt_t<4, 2>(p, u, colour, blocks, pf_stride, st, what, out)
                           : thread_dt_t<4, 4>(p, u, colour, blocks, pf_stride, st, what, out);
        case 5: return two ? thread_dt_t<5, 2>(p, u, colour, blocks, pf_stride, st, what, out)
                           : thread_dt_t<5, 4>(p, u, colour, blocks, pf_stride, st, what, out);
        case 6: return two ? thread_dt_t<6, 2>(p, u, colour, blocks, pf_stride, st, what, out)
                           : thread_dt_t<6, 4>(p, u, colour, blocks, pf_stride, st, what, out);
        default: return cudaErrorInvalidValue;
    }
}

bool thread_dt_supported(const Params &p) { return p.lgS >= 3 && p.lgS <= 6 && p.N <= 7; }

size_t thread_dt_smem(const Params &p)
{
    size_t sm = 0;
    thread_dispatch(p, 0, 0, 0, 0, nullptr, 0, &sm);
    return sm;
}

cudaError_t thread_dt_configure(const Params &p) { return thread_dispatch(p, 0, 0, 0, 0, nullptr, 1, nullptr); }

// One block per tile set (the hardware block scheduler balances sets of unequal duration better
// than a static stride).  pf_stride = resident blocks of the device: when block b is running, block
// b + pf_stride is (about) the one that will take over its slot, so that is the set b prefetches.
cudaError_t thread_dt_grid(const Params &p, int sm_count, uint32_t *blocks, uint32_t *pf_stride)
{
    const uint32_t T = p.L >> p.lgS, half = T >> 1;
    const uint64_t tiles = (uint64_t)p.R * half * half;
    const uint64_t nsets = (tiles + 31) / 32;
    size_t per_sm = 0;
    const cudaError_t e = thread_dispatch(p, 0, 0, 0, 0, nullptr, 3, &per_sm);
    if (e != cudaSuccess) return e;
    if (per_sm == 0) return cudaErrorLaunchOutOfResources;
    const uint64_t slots = (uint64_t)sm_count * per_sm;
    *blocks = (uint32_t)nsets;
    *pf_stride = nsets > slots ? (uint32_t)slots : 0u;
    return cudaSuccess;
}

cudaError_t thread_dt_launch(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, uint32_t pf_stride,
                             cudaStream_t st)
{
    return thread_dispatch(p, u, colour, blocks, pf_stride, st, 2, nullptr);
}

}  // namespace rsos
