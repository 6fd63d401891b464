// rsos_pack.cu -- the packed working lattice of the THREAD engine and its conversion kernels.
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// Under Eq. (6) nearest-neighbour heights differ by at most N, so a surface is fully
// described by its heights mod 2^FB (2^FB > 2N) plus ONE absolute number per realization.  The
// THREAD engine therefore keeps its working state in HBM as FB bits per site (D:5):
//     pk[r][y][w], w < L*FB/32: sites x = w*SPW .. w*SPW+SPW-1 (SPW = 32/FB), site k at bits
//     [k*FB, (k+1)*FB), value h(x, y) mod 2^FB,
// and the exposed int32 heights h[r][y][x] are rebuilt from it on demand (rsos_width, rsos_sums,
// rsos_get_heights, ...):
//     rel(x, y) = V(y) + H(x, y),  V = difference chain down column 0,  H = chain along row y,
//     h(x, y)   = h00 + rel(x, y), h00 = (S1 - sum rel) / L^2,  S1 = sum h = s1off + accepted
// (every accepted deposit adds exactly 1 to sum h; s1off is fixed when the packed copy is made).
// All sums are exact integers; the division must be exact, otherwise ERR_RECONSTRUCT is raised.
#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace rsos {

template <int FB>
__device__ __forceinline__ int32_t sdiff(uint32_t a, uint32_t b)      // sext((a - b) mod 2^FB)
{
    return ((int32_t)((a - b) << (32 - FB))) >> (32 - FB);
}

// ---------------------------------------------------------------------------------------------
// int32 -> packed: one thread per packed word.
// ---------------------------------------------------------------------------------------------
template <int FB>
__global__ void __launch_bounds__(256) pack_kernel(const int32_t *__restrict__ h, uint32_t *__restrict__ pk, size_t nwords)
{
    constexpr uint32_t SPW = 32 / FB, M = (1u << FB) - 1u;
    const size_t w = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= nwords) return;
    const int4 *src = reinterpret_cast<const int4 *>(h + w * SPW);
    uint32_t out = 0;
#pragma unroll
    for (uint32_t c = 0; c < SPW / 4; ++c) {
        const int4 q = src[c];
        const uint32_t v = ((uint32_t)q.x & M) | (((uint32_t)q.y & M) << FB) | (((uint32_t)q.z & M) << (2 * FB)) |
                           (((uint32_t)q.w & M) << (3 * FB));
        out |= v << (c * 4 * FB);
    }
    pk[w] = out;
}

// s1off[r] = S1[r] - accepted[r], S1 from the sums kernel (red[4r] holds S1 as int64 bits).
__global__ void s1off_kernel(const unsigned long long *red, const unsigned long long *accepted, long long *s1off, uint32_t R)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < R) s1off[r] = (long long)red[4 * (size_t)r] - (long long)accepted[r];
}

// ---------------------------------------------------------------------------------------------
// block-wide inclusive scan of one int per thread (256 threads); returns the scan value and the
// block total through *total.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int32_t block_scan_256(int32_t v, int32_t *total, int32_t *sh /* 9 ints */)
{
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int32_t n = __shfl_up_sync(0xFFFFFFFFu, v, o);
        if ((int)lane >= o) v += n;
    }
    __syncthreads();                                   // sh may still be read from a previous call
    if (lane == 31) sh[warp] = v;
    __syncthreads();
    if (warp == 0) {
        int32_t t = lane < 8 ? sh[lane] : 0;
#pragma unroll
        for (int o = 1; o < 8; o <<= 1) {
            const int32_t n = __shfl_up_sync(0xFFFFFFFFu, t, o);
            if ((int)lane >= o) t += n;
        }
        if (lane < 8) sh[lane] = t;                    // inclusive warp totals
        if (lane == 7) sh[8] = t;
    }
    __syncthreads();
    if (warp > 0) v += sh[warp - 1];
    *total = sh[8];
    return v;
}

// V[r][y] = h(0, y) - h(0, 0): chain down column 0.  One block per realization.
template <int FB>
__global__ void __launch_bounds__(256) unpack_col_kernel(const uint32_t *__restrict__ pk, int32_t *__restrict__ V,
                                                         uint32_t L, uint32_t wpr)
{
    constexpr uint32_t M = (1u << FB) - 1u;
    __shared__ int32_t sh[9];
    const uint32_t *base = pk + (size_t)blockIdx.x * L * wpr;
    int32_t carry = 0;
    for (uint32_t y0 = 0; y0 < L; y0 += 256) {
        const uint32_t y = y0 + threadIdx.x;
        int32_t d = 0;
        if (y > 0 && y < L) d = sdiff<FB>(base[(size_t)y * wpr] & M, base[(size_t)(y - 1) * wpr] & M);
        int32_t total;
        const int32_t s = block_scan_256(d, &total, sh);
        if (y < L) V[(size_t)blockIdx.x * L + y] = carry + s;
        carry += total;
    }
}

// ---------------------------------------------------------------------------------------------
// Row chains.  A row of wpr packed words is handled by a TEAM: the whole block (256 threads) when
// wpr >= 256, else one warp (8 rows per block).  Every thread owns a contiguous run of words,
// sums its differences, the team scans the totals, and a second sweep over the same words forms
// rel(x, y) = V(y) + H(x, y) site by site.
//   WRITE = false: srel[4r + 0] += sum_x rel, srel[4r + 1] += sum_x rel^2 (exact, 64-bit),
//                  srel[4r + 2] = min rel, srel[4r + 3] = max rel (signed 64-bit)
//   WRITE = true : h[r][y][x] = h00[r] + rel(x, y)            (int4 stores)
// ---------------------------------------------------------------------------------------------
template <int FB, bool WRITE>
__global__ void __launch_bounds__(256) unpack_rows_kernel(const uint32_t *__restrict__ pk, const int32_t *__restrict__ V,
                                                          const int32_t *__restrict__ h00, int32_t *__restrict__ h,
                                                          unsigned long long *__restrict__ srel, uint32_t L,
                                                          uint32_t wpr, uint32_t nrows)
{
    constexpr uint32_t SPW = 32 / FB, M = (1u << FB) - 1u;
    __shared__ int32_t sh[9];
    const bool team_block = wpr >= 256u;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t row = team_block ? blockIdx.x : blockIdx.x * 8u + warp;
    const bool row_ok = row < nrows;                               // warp-uniform
    const uint32_t tteam = team_block ? threadIdx.x : lane;
    const uint32_t wpt = team_block ? wpr / 256u : (wpr >= 32u ? wpr / 32u : 1u);
    const uint32_t w0 = tteam * wpt;
    const uint32_t nw = (row_ok && w0 < wpr) ? wpt : 0u;
    const uint32_t *rowp = pk + (size_t)(row_ok ? row : 0u) * wpr;
    const uint32_t rl = (row_ok ? row : 0u) / L;

    // phase 1: total of my differences (site 0 of the row has difference 0: H(0, y) = 0)
    uint32_t prevf = 0;
    if (nw) prevf = (w0 == 0u) ? (rowp[0] & M) : (rowp[w0 - 1u] >> (32 - FB));
    int32_t tot = 0;
    {
        uint32_t pf = prevf;
        for (uint32_t i = 0; i < nw; ++i) {
            const uint32_t w = rowp[w0 + i];
#pragma unroll
            for (uint32_t k = 0; k < SPW; ++k) {
                const uint32_t f = (w >> (k * FB)) & M;
                tot += sdiff<FB>(f, pf);
                pf = f;
            }
        }
    }
    int32_t incl;
    if (team_block) {
        int32_t total;
        incl = block_scan_256(tot, &total, sh);
    } else {
        incl = tot;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int32_t n = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if ((int)lane >= o) incl += n;
        }
    }
    // phase 2
    int32_t run = incl - tot;
    if (row_ok) run += V[row];
    if (WRITE && row_ok) run += h00[rl];
    long long acc = 0;
    unsigned long long acc2 = 0;
    int32_t mn = 0x7FFFFFFF, mx = -0x7FFFFFFF - 1;
    {
        uint32_t pf = prevf;
        for (uint32_t i = 0; i < nw; ++i) {
            const uint32_t w = rowp[w0 + i];
            int32_t out[SPW];
#pragma unroll
            for (uint32_t k = 0; k < SPW; ++k) {
                const uint32_t f = (w >> (k * FB)) & M;
                run += sdiff<FB>(f, pf);
                pf = f;
                out[k] = run;
                if (!WRITE) {
                    acc += run;
                    acc2 += (unsigned long long)((long long)run * run);
                    mn = min(mn, run);
                    mx = max(mx, run);
                }
            }
            if (WRITE) {
                int4 *dst = reinterpret_cast<int4 *>(h + (size_t)row * L + (size_t)(w0 + i) * SPW);
#pragma unroll
                for (uint32_t c = 0; c < SPW / 4; ++c)
                    dst[c] = make_int4(out[4 * c], out[4 * c + 1], out[4 * c + 2], out[4 * c + 3]);
            }
        }
    }
    if (!WRITE) {
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
            acc2 += __shfl_xor_sync(0xFFFFFFFFu, acc2, o);
            mn = min(mn, __shfl_xor_sync(0xFFFFFFFFu, mn, o));
            mx = max(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, o));
        }
        // The rows of one block belong to one realization whenever a realization has at least 8 rows (L >= 8, always):
        // team_block: one row; else 8 consecutive rows, and L is a multiple of 8.  Reduce over the 8 warps first so
        // that a block sends ONE set of atomics (they all land on the four words of its realization).
        __shared__ long long b_acc[8];
        __shared__ unsigned long long b_acc2[8];
        __shared__ int32_t b_mn[8], b_mx[8];
        if (lane == 0) {
            b_acc[warp] = row_ok ? acc : 0;
            b_acc2[warp] = row_ok ? acc2 : 0ull;
            b_mn[warp] = row_ok ? mn : 0x7FFFFFFF;
            b_mx[warp] = row_ok ? mx : -0x7FFFFFFF - 1;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            const uint32_t row0 = team_block ? blockIdx.x : blockIdx.x * 8u;
            if (row0 < nrows) {
                long long a = 0;
                unsigned long long a2 = 0;
                int32_t lo = 0x7FFFFFFF, hi = -0x7FFFFFFF - 1;
#pragma unroll
                for (int w = 0; w < 8; ++w) { a += b_acc[w]; a2 += b_acc2[w]; lo = min(lo, b_mn[w]); hi = max(hi, b_mx[w]); }
                unsigned long long *d = srel + 4 * (size_t)(row0 / L);
                if (a != 0) atomicAdd(d, (unsigned long long)a);
                if (a2 != 0) atomicAdd(d + 1, a2);
                if (lo <= hi) {
                    atomicMin(reinterpret_cast<long long *>(d + 2), (long long)lo);
                    atomicMax(reinterpret_cast<long long *>(d + 3), (long long)hi);
                }
            }
        }
    }
}

__global__ void srel_init_kernel(unsigned long long *srel, uint32_t R)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    srel[4 * (size_t)r] = 0ull;
    srel[4 * (size_t)r + 1] = 0ull;
    srel[4 * (size_t)r + 2] = (unsigned long long)0x7FFFFFFFFFFFFFFFll;
    srel[4 * (size_t)r + 3] = (unsigned long long)(-0x7FFFFFFFFFFFFFFFll - 1);
}

// h00[r] = (s1off[r] + accepted[r] - srel[4r]) / L^2, which must divide exactly and fit int32.
__global__ void anchor_kernel(const long long *s1off, const unsigned long long *accepted, const unsigned long long *srel,
                              int32_t *h00, uint32_t lgL2, uint32_t R, uint32_t *err)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    const long long num = s1off[r] + (long long)accepted[r] - (long long)srel[4 * (size_t)r];
    const long long q = num >> lgL2;
    if ((q << lgL2) != num || q > 0x7FFFFFFFll || q < -0x80000000ll) atomicOr(err, ERR_RECONSTRUCT);
    h00[r] = (int32_t)q;
}

// =============================================================================================
// General L (D:2b): the same packed format with a row pitch of wpr = ceil(L * FB / 32) words; site x of a row sits in
// word x / SPW at bit (x mod SPW) * FB, the bits of the last word beyond site L - 1 are unused.  The kernels below are
// the plain forms of the ones above (no int4 accesses, no power-of-two shifts): one thread per packed word, one warp
// per row.  They are used only when L is not a power of two.
// =============================================================================================
template <int FB>
__global__ void __launch_bounds__(256) gpack_kernel(const int32_t *__restrict__ h, uint32_t *__restrict__ pk, uint32_t L,
                                                    uint32_t wpr, size_t nwords)
{
    constexpr uint32_t SPW = 32 / FB, M = (1u << FB) - 1u;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nwords) return;
    const size_t row = i / wpr;
    const uint32_t w = (uint32_t)(i - row * wpr);
    const int32_t *src = h + row * L;
    uint32_t out = 0;
#pragma unroll
    for (uint32_t k = 0; k < SPW; ++k) {
        const uint32_t x = w * SPW + k;
        if (x < L) out |= ((uint32_t)src[x] & M) << (k * FB);
    }
    pk[i] = out;
}

template <int FB, bool WRITE>
__global__ void __launch_bounds__(256) gunpack_rows_kernel(const uint32_t *__restrict__ pk, const int32_t *__restrict__ V,
                                                           const int32_t *__restrict__ h00, int32_t *__restrict__ h,
                                                           unsigned long long *__restrict__ srel, uint32_t L, uint32_t wpr,
                                                           uint32_t nrows)
{
    constexpr uint32_t SPW = 32 / FB, M = (1u << FB) - 1u;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t row = blockIdx.x * 8u + warp;
    const bool row_ok = row < nrows;                               // warp-uniform
    const uint32_t wpt = (wpr + 31u) / 32u;
    const uint32_t w0 = lane * wpt;
    const uint32_t nw = (row_ok && w0 < wpr) ? min(wpt, wpr - w0) : 0u;
    const uint32_t *rowp = pk + (size_t)(row_ok ? row : 0u) * wpr;
    const uint32_t rl = (row_ok ? row : 0u) / L;

    uint32_t prevf = 0;                                            // the field before my first site (site 0: itself)
    if (nw) prevf = (w0 == 0u) ? (rowp[0] & M) : (rowp[w0 - 1u] >> (32 - FB));
    int32_t tot = 0;
    {
        uint32_t pf = prevf;
        for (uint32_t i = 0; i < nw; ++i) {
            const uint32_t w = rowp[w0 + i];
#pragma unroll
            for (uint32_t k = 0; k < SPW; ++k) {
                if ((w0 + i) * SPW + k < L) {
                    const uint32_t f = (w >> (k * FB)) & M;
                    tot += sdiff<FB>(f, pf);
                    pf = f;
                }
            }
        }
    }
    int32_t incl = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int32_t n = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if ((int)lane >= o) incl += n;
    }
    int32_t run = incl - tot;
    if (row_ok) run += V[row];
    if (WRITE && row_ok) run += h00[rl];
    long long acc = 0;
    unsigned long long acc2 = 0;
    int32_t mn = 0x7FFFFFFF, mx = -0x7FFFFFFF - 1;
    {
        uint32_t pf = prevf;
        for (uint32_t i = 0; i < nw; ++i) {
            const uint32_t w = rowp[w0 + i];
#pragma unroll
            for (uint32_t k = 0; k < SPW; ++k) {
                const uint32_t x = (w0 + i) * SPW + k;
                if (x < L) {
                    const uint32_t f = (w >> (k * FB)) & M;
                    run += sdiff<FB>(f, pf);
                    pf = f;
                    if (WRITE) h[(size_t)row * L + x] = run;
                    else {
                        acc += run;
                        acc2 += (unsigned long long)((long long)run * run);
                        mn = min(mn, run);
                        mx = max(mx, run);
                    }
                }
            }
        }
    }
    if (!WRITE) {
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
            acc2 += __shfl_xor_sync(0xFFFFFFFFu, acc2, o);
            mn = min(mn, __shfl_xor_sync(0xFFFFFFFFu, mn, o));
            mx = max(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, o));
        }
        if (lane == 0 && row_ok) {                                  // a block's 8 rows may belong to two realizations: per warp
            unsigned long long *d = srel + 4 * (size_t)rl;
            if (acc != 0) atomicAdd(d, (unsigned long long)acc);
            if (acc2 != 0) atomicAdd(d + 1, acc2);
            if (mn <= mx) {
                atomicMin(reinterpret_cast<long long *>(d + 2), (long long)mn);
                atomicMax(reinterpret_cast<long long *>(d + 3), (long long)mx);
            }
        }
    }
}

// h00[r] = (s1off[r] + accepted[r] - srel[4r]) / L^2 for any L; must divide exactly and fit int32.
__global__ void ganchor_kernel(const long long *s1off, const unsigned long long *accepted, const unsigned long long *srel,
                               int32_t *h00, long long n2, uint32_t R, uint32_t *err)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    const long long num = s1off[r] + (long long)accepted[r] - (long long)srel[4 * (size_t)r];
    const long long q = num / n2;
    if (q * n2 != num || q > 0x7FFFFFFFll || q < -0x80000000ll) atomicOr(err, ERR_RECONSTRUCT);
    h00[r] = (int32_t)q;
}

// =============================================================================================
// Host-side launchers
// =============================================================================================
cudaError_t launch_pack(const Params &p, cudaStream_t st)
{
    if (p.general) {
        const uint32_t wpr = (p.L * p.FB + 31u) / 32u;
        const size_t nw = (size_t)p.R * p.L * wpr;
        const uint32_t gb = (uint32_t)((nw + 255) / 256);
        if (p.FB == 2) gpack_kernel<2><<<gb, 256, 0, st>>>(p.h, p.pk, p.L, wpr, nw);
        else gpack_kernel<4><<<gb, 256, 0, st>>>(p.h, p.pk, p.L, wpr, nw);
        return cudaGetLastError();
    }
    const size_t nwords = (size_t)p.R * p.L * p.L * p.FB / 32;
    const uint32_t blocks = (uint32_t)((nwords + 255) / 256);
    if (p.FB == 2) pack_kernel<2><<<blocks, 256, 0, st>>>(p.h, p.pk, nwords);
    else pack_kernel<4><<<blocks, 256, 0, st>>>(p.h, p.pk, nwords);
    return cudaGetLastError();
}

cudaError_t launch_s1off(const Params &p, const unsigned long long *d_red, long long *d_s1off, cudaStream_t st)
{
    s1off_kernel<<<(p.R + 127) / 128, 128, 0, st>>>(d_red, p.accepted, d_s1off, p.R);
    return cudaGetLastError();
}

// Sums of the relative heights straight from the packed lattice: d_srel[4r..4r+3] = sum rel,
// sum rel^2, min rel, max rel (rel = h - h(0,0)).  Enough for S1, S2 and max |h| without
// materialising the int32 heights.  Scratch: d_V (R*L int32).  3 kernels.
cudaError_t launch_packed_sums(const Params &p, int32_t *d_V, unsigned long long *d_srel, cudaStream_t st)
{
    if (p.general) {
        const uint32_t gwpr = (p.L * p.FB + 31u) / 32u, gnrows = p.R * p.L;
        srel_init_kernel<<<(p.R + 127) / 128, 128, 0, st>>>(d_srel, p.R);
        if (p.FB == 2) {
            unpack_col_kernel<2><<<p.R, 256, 0, st>>>(p.pk, d_V, p.L, gwpr);
            gunpack_rows_kernel<2, false><<<(gnrows + 7u) / 8u, 256, 0, st>>>(p.pk, d_V, nullptr, p.h, d_srel, p.L, gwpr, gnrows);
        } else {
            unpack_col_kernel<4><<<p.R, 256, 0, st>>>(p.pk, d_V, p.L, gwpr);
            gunpack_rows_kernel<4, false><<<(gnrows + 7u) / 8u, 256, 0, st>>>(p.pk, d_V, nullptr, p.h, d_srel, p.L, gwpr, gnrows);
        }
        return cudaGetLastError();
    }
    const uint32_t wpr = p.L * p.FB / 32;
    const uint32_t nrows = p.R * p.L;
    const uint32_t rblocks = wpr >= 256u ? nrows : (nrows + 7u) / 8u;
    srel_init_kernel<<<(p.R + 127) / 128, 128, 0, st>>>(d_srel, p.R);
    if (p.FB == 2) {
        unpack_col_kernel<2><<<p.R, 256, 0, st>>>(p.pk, d_V, p.L, wpr);
        unpack_rows_kernel<2, false><<<rblocks, 256, 0, st>>>(p.pk, d_V, nullptr, p.h, d_srel, p.L, wpr, nrows);
    } else {
        unpack_col_kernel<4><<<p.R, 256, 0, st>>>(p.pk, d_V, p.L, wpr);
        unpack_rows_kernel<4, false><<<rblocks, 256, 0, st>>>(p.pk, d_V, nullptr, p.h, d_srel, p.L, wpr, nrows);
    }
    return cudaGetLastError();
}

// packed -> int32 heights of all realizations.  Scratch: d_V (R*L int32), d_srel (4R uint64),
// d_h00 (R int32).  Returns the number of kernels launched through *launches.
cudaError_t launch_unpack(const Params &p, const long long *d_s1off, int32_t *d_V, unsigned long long *d_srel,
                          int32_t *d_h00, cudaStream_t st, uint32_t *launches)
{
    const uint32_t wpr = p.L * p.FB / 32;
    const uint32_t nrows = p.R * p.L;
    const uint32_t rblocks = wpr >= 256u ? nrows : (nrows + 7u) / 8u;
    cudaError_t e = launch_packed_sums(p, d_V, d_srel, st);
    if (e != cudaSuccess) return e;
    if (p.general) {
        const uint32_t gwpr = (p.L * p.FB + 31u) / 32u;
        ganchor_kernel<<<(p.R + 127) / 128, 128, 0, st>>>(d_s1off, p.accepted, d_srel, d_h00, (long long)p.L * p.L, p.R, p.err);
        if (p.FB == 2) gunpack_rows_kernel<2, true><<<(nrows + 7u) / 8u, 256, 0, st>>>(p.pk, d_V, d_h00, p.h, d_srel, p.L, gwpr, nrows);
        else gunpack_rows_kernel<4, true><<<(nrows + 7u) / 8u, 256, 0, st>>>(p.pk, d_V, d_h00, p.h, d_srel, p.L, gwpr, nrows);
        *launches = 5;
        return cudaGetLastError();
    }
    anchor_kernel<<<(p.R + 127) / 128, 128, 0, st>>>(d_s1off, p.accepted, d_srel, d_h00, 2 * p.lgL, p.R, p.err);
    if (p.FB == 2) unpack_rows_kernel<2, true><<<rblocks, 256, 0, st>>>(p.pk, d_V, d_h00, p.h, d_srel, p.L, wpr, nrows);
    else unpack_rows_kernel<4, true><<<rblocks, 256, 0, st>>>(p.pk, d_V, d_h00, p.h, d_srel, p.L, wpr, nrows);
    *launches = 5;
    return cudaGetLastError();
}

}  // namespace rsos
