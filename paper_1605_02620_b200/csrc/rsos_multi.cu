// rsos_multi.cu -- the MULTI engine: the paper's shared-coordinate multisurface layout (sm_100a).
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// "Each single instruction multiple thread (SIMT) unit of the GPU updates 128 realizations, in which the
// sequence of randomly selected coordinates for update is the same.  This correlation was broken by updating only
// half of the selected lattice sites in each attempt."  Schedule MS of D:2d (reading Q5): realizations are grouped
// by global index, group g = r div 128; in sweep t the group draws 2 L^2 coordinates in order from
// Philox(q, 0xFFFFFFFD, t, g) (slot layout of RS, D:2 step 6) and member b = r mod 128 attempts selection a iff
// bit (b mod 32) of word (b div 32) of Philox(a, 0xFFFFFFFC, t, g) is 1.
//
// One warp = 32 consecutive members of a group = one block.  The surfaces of the warp live in shared memory with
// the REALIZATION INNERMOST, element (site, lane): every one of the five loads and the store of an attempt touches
// 32 consecutive elements -- coalesced and conflict-free by construction, which is the point of the paper's layout
// -- and the site and its address are warp-uniform.  Elements are int16 heights relative to the surface's own
// h(0,0) at the start of the launch: |h(x) - h(0,0)| <= 2 N L on a surface that satisfies Eq. (6), and a launch of
// M MCS raises a site by at most 2 M + 2 N L, so with M <= 4096, N <= 31, L <= 32 everything stays below 2^15.
#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace rsos {

__global__ void __launch_bounds__(32) multi_rs_kernel(Params p, uint32_t t0, uint32_t mcs)
{
    extern __shared__ __align__(16) uint32_t smem[];
    int16_t *lat = reinterpret_cast<int16_t *>(smem);               // [site][lane]
    const uint32_t lane = threadIdx.x;
    const uint32_t L = p.L, Lm = L - 1u, lgL = p.lgL, n = L * L;
    const uint32_t rl = blockIdx.x * 32u + lane;
    const bool live = rl < p.R;
    const uint32_t rg0 = p.first_real + blockIdx.x * 32u;            // first member of this warp (a multiple of 32)
    const uint32_t g = rg0 >> 7, wsel = (rg0 >> 5) & 3u;             // group, mask word of this warp
    int32_t *h = p.h + (size_t)(live ? rl : 0u) * n;
    const int32_t ref = live ? h[0] : 0;
    for (uint32_t s = 0; s < n; ++s) lat[s * 32u + lane] = live ? (int16_t)(h[s] - ref) : (int16_t)0;
    __syncwarp();

    const int32_t N = (int32_t)p.N;
    const uint32_t A = 2u * n;
    uint32_t nacc = 0;
    for (uint32_t m = 0; m < mcs; ++m) {
        const uint32_t t = t0 + m;
#pragma unroll 1
        for (uint32_t q = 0; q < A / 8u; ++q) {
            const uint4 co = philox4x32_10(q, 0xFFFFFFFDu, t, g, p.k0, p.k1);      // 8 coordinates (2 lg L <= 16)
            const uint32_t cw[4] = {co.x, co.y, co.z, co.w};
#pragma unroll
            for (uint32_t w = 0; w < 8; ++w) {
                const uint32_t v = (w & 1u) ? cw[w >> 1] >> 16 : cw[w >> 1];
                const uint32_t x = v & Lm, y = (v >> lgL) & Lm;
                const uint4 mo = philox4x32_10(q * 8u + w, 0xFFFFFFFCu, t, g, p.k0, p.k1);
                const uint32_t mw = wsel == 0u ? mo.x : wsel == 1u ? mo.y : wsel == 2u ? mo.z : mo.w;
                const bool take = ((mw >> lane) & 1u) != 0u;
                int16_t *row = lat + ((y << lgL) * 32u + lane);
                const int32_t c = (int32_t)row[x * 32u] + 1;
                const int32_t l = row[((x - 1u) & Lm) * 32u], r = row[((x + 1u) & Lm) * 32u];
                const int32_t up = lat[((((y - 1u) & Lm) << lgL) + x) * 32u + lane];
                const int32_t dn = lat[((((y + 1u) & Lm) << lgL) + x) * 32u + lane];
                const bool ok = take && abs(c - l) <= N && abs(c - r) <= N && abs(c - up) <= N && abs(c - dn) <= N;
                if (ok) row[x * 32u] = (int16_t)c;
                nacc += ok ? 1u : 0u;
            }
        }
    }
    __syncwarp();
    if (live) {
        for (uint32_t s = 0; s < n; ++s) h[s] = ref + (int32_t)lat[s * 32u + lane];
        if (nacc) atomicAdd(p.accepted + rl, (unsigned long long)nacc);
    }
}

// RS mode on a power-of-two lattice of at most 32 x 32 sites, N <= 31, first_real a multiple of 32 (a warp's 32
// members must share their group and their mask word).
bool multi_ok(uint32_t L, uint32_t N, uint32_t first_real) { return L <= 32 && N <= 31 && first_real % 32u == 0; }
size_t multi_smem(const Params &p) { return (size_t)p.L * p.L * 32 * sizeof(int16_t); }
uint32_t multi_blocks(const Params &p) { return (p.R + 31u) / 32u; }
cudaError_t multi_configure(const Params &p)
{
    return cudaFuncSetAttribute(multi_rs_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)multi_smem(p));
}
cudaError_t multi_launch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st)
{
    multi_rs_kernel<<<multi_blocks(p), 32, multi_smem(p), st>>>(p, t0, mcs);
    return cudaGetLastError();
}

}  // namespace rsos
