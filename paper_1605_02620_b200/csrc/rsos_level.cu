// rsos_level.cu -- the LEVEL engine: serial random-sequential deposition (RS mode) of FEW realizations (sm_100a).
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// In RS mode (2S > L, D:2 step 3) the L*L attempts of an MCS of one realization form one sequential chain, and
// BASELINE configs[0] has only 128 realizations: 128 chains cannot fill a B200, whatever a warp does with a window of
// 32 attempts (ONCHIP engine: about 10 of 32 committed per window on a 1024-site lattice).  But two attempts interact
// only if their sites are EQUAL OR NEAREST NEIGHBOURS: attempt j reads its site and the four neighbours and writes its
// site, so it depends on an earlier attempt i exactly when site(i) lies in the 5-point stencil of site(j) (and then,
// adjacency being symmetric, i also reads what j writes).  Executing a batch of B consecutive attempts in DEPENDENCY
// LEVELS -- an attempt runs as soon as no earlier unfinished attempt of the batch sits in its stencil -- gives exactly
// the sequential result, and a batch of 256 attempts on a 32 x 32 lattice is only a few levels deep.
//
// One block per realization, thread j owns attempt a0 + j of the current batch.  The whole lattice lives in shared
// memory (one byte per site, height mod 256: N <= 127 keeps every nearest-neighbour difference recoverable) for all
// MCS of the call.  Per round r of a batch:
//   1. every unfinished thread claims its site:  atomicMax(own[site], (r << 10) | (1023 - j))  -- the round stamp
//      makes claims of earlier rounds lose, within a round the SMALLEST j wins;
//   2. barrier;
//   3. a thread is READY iff none of the five entries of its stencil carries a claim of THIS round by a smaller j
//      (for its own site: the claim is its own).  Two ready attempts are never equal or adjacent: each would need
//      the smaller index.  Ready threads apply Eq. (6) to their stencil and store; they are finished;
//   4. barrier with OR-reduction: any thread unfinished -> next round.
// (Posting the next round's claim early into a second table, one barrier per round, was measured: slower.)
// The int32 heights are rebuilt at the end from difference chains and sum h = sum h0 + accepted, as in the ONCHIP
// engine (D:4, D:5).
#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace rsos {

constexpr uint32_t LEVEL_B = 512;            // attempts in flight per realization = threads per block

__device__ __forceinline__ int32_t sext8(uint32_t d) { return (int32_t)(int8_t)(d & 0xFFu); }

__global__ void __launch_bounds__(LEVEL_B) level_rs_kernel(Params p, uint32_t t0, uint32_t mcs)
{
    extern __shared__ __align__(16) uint32_t smem[];
    const uint32_t L = p.L, Lm = L - 1u, lgL = p.lgL, n = L * L;
    uint32_t *own = smem;                                              // n words: claims
    uint8_t *hb = reinterpret_cast<uint8_t *>(smem + n);               // n bytes: heights mod 256
    uint32_t *tab = smem + n + n / 4u;                            // 2 x (Philox calls of a batch, 16 B each)
    __shared__ long long red[LEVEL_B / 32];
    __shared__ long long bcast;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t rl = blockIdx.x;
    const uint32_t rg = p.first_real + rl;
    int32_t *h = p.h + (size_t)rl * n;

    // ---- stage the lattice; S1 = sum of the int32 heights (exact) ---------------------------------------------------
    long long s1 = 0;
    for (uint32_t i = tid; i < n; i += LEVEL_B) {
        const int32_t v = h[i];
        s1 += v;
        hb[i] = (uint8_t)((uint32_t)v & 0xFFu);
    }
    __syncthreads();

    const bool w16 = 2u * lgL <= 16u;                                   // D:2 step 6: 16-bit slots while 2 lg L <= 16
    const uint32_t lg_ns = w16 ? 3u : 2u;
    const uint32_t ncall = LEVEL_B >> lg_ns;                            // Philox calls per batch
    const uint32_t nbatch = (n + LEVEL_B - 1u) / LEVEL_B;
    const int32_t N = (int32_t)p.N;
    uint32_t nacc = 0;
    // calls of batch b of sweep t -> tab buffer (b & 1): attempt a takes slot a mod ns of call a div ns
    auto fill = [&](uint32_t t, uint32_t b) {
        if (tid < ncall)
            reinterpret_cast<uint4 *>(tab)[(b & 1u) * ncall + tid] = philox4x32_10(b * ncall + tid, 0u, t, rg, p.k0, p.k1);
    };
    for (uint32_t i = tid; i < n; i += LEVEL_B) own[i] = 0u;
    uint32_t rnd = 0;                                                   // rounds since the last reset of the claim tables
    for (uint32_t m = 0; m < mcs; ++m) {
        const uint32_t t = t0 + m;
        if (rnd > (1u << 21)) {                                         // keep the round stamp inside its 22 bits
            __syncthreads();
            for (uint32_t i = tid; i < n; i += LEVEL_B) own[i] = 0u;
            rnd = 0;
        }
        fill(t, 0u);
        __syncthreads();
        for (uint32_t b = 0; b < nbatch; ++b) {
            const uint32_t a = b * LEVEL_B + tid;
            bool todo = a < n;
            uint32_t v;
            if (w16) v = reinterpret_cast<const uint16_t *>(tab + (b & 1u) * ncall * 4u)[tid];   // halfword tid of the batch
            else v = tab[(b & 1u) * ncall * 4u + tid];
            if (b + 1u < nbatch) fill(t, b + 1u);                       // the next batch's calls, off the critical path
            const uint32_t x = v & Lm, y = (v >> lgL) & Lm;
            const uint32_t sC = (y << lgL) + x;
            const uint32_t sL = (y << lgL) + ((x - 1u) & Lm), sR = (y << lgL) + ((x + 1u) & Lm);
            const uint32_t sU = (((y - 1u) & Lm) << lgL) + x, sD = (((y + 1u) & Lm) << lgL) + x;
            const uint32_t mine = 1023u - tid;
            int any = 1;
            while (any) {
                ++rnd;
                const uint32_t claim = (rnd << 10) | mine;
                if (todo) atomicMax(own + sC, claim);
                __syncthreads();
                if (todo) {
                    // the stencil's heights are loaded together with its claims (harmless if the thread turns out
                    // blocked; stable if it is ready: no ready attempt is equal or adjacent to another one)
                    const uint32_t oC = own[sC], oL = own[sL], oR = own[sR], oU = own[sU], oD = own[sD];
                    const uint32_t hC = hb[sC], hL = hb[sL], hR = hb[sR], hU = hb[sU], hD = hb[sD];
                    // blocked by a claim of this round with a smaller attempt index (= a larger low field)
                    const bool ready = oC == claim && !(oL > claim) && !(oR > claim) && !(oU > claim) && !(oD > claim);
                    const uint32_t c = hC + 1u;
                    const bool ok = abs(sext8(c - hL)) <= N && abs(sext8(c - hR)) <= N && abs(sext8(c - hU)) <= N &&
                                    abs(sext8(c - hD)) <= N;
                    if (ready & ok) { hb[sC] = (uint8_t)c; ++nacc; }
                    if (ready) todo = false;
                }
                any = __syncthreads_or(todo ? 1 : 0);
            }
        }
    }
    __syncthreads();

    // ---- accepted deposits of the block ---------------------------------------------------------------------------
    auto block_sum = [&](long long v) -> long long {
        for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
        __syncthreads();
        if (lane == 0) red[warp] = v;
        __syncthreads();
        if (tid == 0) { long long s = 0; for (uint32_t w = 0; w < LEVEL_B / 32; ++w) s += red[w]; bcast = s; }
        __syncthreads();
        return bcast;
    };
    const long long tot = block_sum((long long)nacc);
    s1 = block_sum(s1);
    if (tot == 0) return;                                               // nothing deposited: global heights are current

    // ---- rebuild: rel(x, y) = h(x, y) - h(0, 0) by difference chains: row 0 along x, then every column downwards ----
    int32_t *rel0 = reinterpret_cast<int32_t *>(own);                   // reuse: L words
    if (tid == 0) {
        int32_t r = 0;
        rel0[0] = 0;
        for (uint32_t X = 1; X < L; ++X) { r += sext8((uint32_t)hb[X] - (uint32_t)hb[X - 1u]); rel0[X] = r; }
    }
    __syncthreads();
    long long srel = 0;
    for (uint32_t X = tid; X < L; X += LEVEL_B) {
        int32_t rv = rel0[X];
        srel += rv;
        for (uint32_t Y = 1; Y < L; ++Y) {
            rv += sext8((uint32_t)hb[(Y << lgL) + X] - (uint32_t)hb[((Y - 1u) << lgL) + X]);
            srel += rv;
        }
    }
    srel = block_sum(srel);
    // L^2 * h00 + srel = s1 + accepted
    const long long num = s1 + tot - srel;
    const long long h00 = num >> (2u * lgL);
    if ((h00 << (2u * lgL)) != num) { if (tid == 0) atomicOr(p.err, ERR_RECONSTRUCT); return; }
    for (uint32_t X = tid; X < L; X += LEVEL_B) {
        int32_t hv = (int32_t)h00 + rel0[X];
        h[X] = hv;
        for (uint32_t Y = 1; Y < L; ++Y) {
            hv += sext8((uint32_t)hb[(Y << lgL) + X] - (uint32_t)hb[((Y - 1u) << lgL) + X]);
            h[(size_t)(Y << lgL) + X] = hv;
        }
    }
    if (tid == 0) atomicAdd(p.accepted + rl, (unsigned long long)tot);
}

// RS mode on a power-of-two lattice with L*L >= 256 sites whose claims and heights fit in shared memory (L <= 128).
bool level_ok(uint32_t L, uint32_t N) { return L >= 16 && L <= 128 && N <= 127; }
size_t level_smem(const Params &p) { return (size_t)p.L * p.L * 5 + 2 * LEVEL_B * 4; }
uint32_t level_blocks(const Params &p) { return p.R; }
cudaError_t level_configure(const Params &p)
{
    return cudaFuncSetAttribute(level_rs_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)level_smem(p));
}
cudaError_t level_launch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st)
{
    level_rs_kernel<<<level_blocks(p), LEVEL_B, level_smem(p), st>>>(p, t0, mcs);
    return cudaGetLastError();
}

}  // namespace rsos
