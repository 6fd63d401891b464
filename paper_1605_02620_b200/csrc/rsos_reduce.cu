// rsos_reduce.cu -- width reductions (sm_100a).  Product code; shares nothing with oracle/.
//
// Eq. (2): W^2 = (1/L^2) sum h^2 - ((1/L^2) sum h)^2 per realization.  The kernels return
// exact integers S1 = sum h (int64) and S2 = sum h^2 (uint64); the division happens once on the
// host from a 128-bit numerator (rsos_api.cu).  Integer adds commute, so the block order and the
// atomics do not affect the result.  HBM-bound: 4 B per site, int4 loads, grid = multiple of SMs.
#include <mutex>

#include "../../include/rsos.h"
#include "rsos_internal.h"

namespace rsos {

constexpr int RED_THREADS = 256;

// VEC: n is a multiple of 4 sites per surface (every power-of-two lattice), int4 loads; otherwise (general L with
// L*L not a multiple of 4, D:2b) one site per load.
template <bool VEC>
__global__ void __launch_bounds__(RED_THREADS) sums_kernel(const int32_t *__restrict__ h, uint32_t n /* VEC: L*L/4, else L*L */,
                                                           unsigned long long *out)
{
    const uint32_t r = blockIdx.y;
    long long s1 = 0;
    unsigned long long s2 = 0;
    unsigned int mx = 0;
    if (VEC) {
        const int4 *src = reinterpret_cast<const int4 *>(h) + (size_t)r * n;
        for (uint32_t i = blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += gridDim.x * RED_THREADS) {
            const int4 q = __ldg(src + i);
            s1 += (long long)q.x + (long long)q.y + (long long)q.z + (long long)q.w;
            s2 += (unsigned long long)((long long)q.x * q.x) + (unsigned long long)((long long)q.y * q.y) +
                  (unsigned long long)((long long)q.z * q.z) + (unsigned long long)((long long)q.w * q.w);
            mx = max(max(mx, (unsigned int)abs(q.x)), max((unsigned int)abs(q.y), max((unsigned int)abs(q.z), (unsigned int)abs(q.w))));
        }
    } else {
        const int32_t *src = h + (size_t)r * n;
        // 64-bit index: at L = 65535 (the one odd L this large) n = 4294836225 and a 32-bit i + stride would wrap below n
        for (uint64_t i = (uint64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (uint64_t)gridDim.x * RED_THREADS) {
            const int v = __ldg(src + i);
            s1 += (long long)v;
            s2 += (unsigned long long)((long long)v * v);
            mx = max(mx, (unsigned int)abs(v));
        }
    }
    for (int o = 16; o; o >>= 1) {
        s1 += __shfl_xor_sync(0xFFFFFFFFu, s1, o);
        s2 += __shfl_xor_sync(0xFFFFFFFFu, s2, o);
        mx = max(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, o));
    }
    __shared__ long long w1[RED_THREADS / 32];
    __shared__ unsigned long long w2[RED_THREADS / 32];
    __shared__ unsigned int wm[RED_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { w1[warp] = s1; w2[warp] = s2; wm[warp] = mx; }
    __syncthreads();
    if (warp == 0) {
        s1 = lane < RED_THREADS / 32 ? w1[lane] : 0;
        s2 = lane < RED_THREADS / 32 ? w2[lane] : 0;
        mx = lane < RED_THREADS / 32 ? wm[lane] : 0;
        for (int o = 4; o; o >>= 1) {
            s1 += __shfl_xor_sync(0xFFFFFFFFu, s1, o);
            s2 += __shfl_xor_sync(0xFFFFFFFFu, s2, o);
            mx = max(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, o));
        }
        if (lane == 0) {
            atomicAdd(out + 4 * r + 0, (unsigned long long)s1);      // two's complement: exact mod 2^64
            atomicAdd(out + 4 * r + 1, s2);
            atomicMax(out + 4 * r + 2, (unsigned long long)mx);
        }
    }
}

cudaError_t launch_sums(const int32_t *h, uint32_t L, uint32_t R, unsigned long long *d_out, int sm_count, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(d_out, 0, (size_t)R * 4 * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    const bool vec = ((uint64_t)L * L) % 4 == 0;
    const uint64_t n4 = vec ? (uint64_t)L * L / 4 : (uint64_t)L * L;
    // enough blocks per realization to cover every SM with 8 blocks, at most one block per 256*4 loads
    uint64_t bx = (n4 + RED_THREADS * 4 - 1) / (RED_THREADS * 4);
    const uint64_t want = ((uint64_t)(sm_count > 0 ? sm_count : 1) * 8 + R - 1) / R;
    if (bx > want) bx = want;
    if (bx < 1) bx = 1;
    for (uint32_t r0 = 0; r0 < R; r0 += 65535) {
        const uint32_t nr = R - r0 < 65535 ? R - r0 : 65535;
        if (vec) sums_kernel<true><<<dim3((unsigned)bx, nr), RED_THREADS, 0, st>>>(h + (size_t)r0 * L * L, (uint32_t)n4, d_out + 4 * (size_t)r0);
        else sums_kernel<false><<<dim3((unsigned)bx, nr), RED_THREADS, 0, st>>>(h + (size_t)r0 * L * L, (uint32_t)n4, d_out + 4 * (size_t)r0);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ---------------------------------------------------------------------------------------------
// Central power sums about an integer base b[r] (Eq. 13-15): M_k = sum (h - b)^k,
// k = 1..4, exact in 128-bit two's complement.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void add128(unsigned long long *dst, __int128 v)
{
    const unsigned long long lo = (unsigned long long)v, hi = (unsigned long long)(v >> 64);
    const unsigned long long old = atomicAdd(dst, lo);
    const unsigned long long carry = (old + lo < old) ? 1ull : 0ull;
    if (hi + carry) atomicAdd(dst + 1, hi + carry);
}

__device__ __forceinline__ __int128 shfl_xor128(__int128 v, int o)
{
    unsigned long long lo = (unsigned long long)v, hi = (unsigned long long)(v >> 64);
    lo = __shfl_xor_sync(0xFFFFFFFFu, lo, o);
    hi = __shfl_xor_sync(0xFFFFFFFFu, hi, o);
    return (__int128)(((unsigned __int128)hi << 64) | lo);
}

template <bool VEC>
__global__ void __launch_bounds__(RED_THREADS) moments_kernel(const int32_t *__restrict__ h, uint32_t n4,
                                                              const long long *__restrict__ base, unsigned long long *out)
{
    const uint32_t r = blockIdx.y;
    const long long b = base[r];
    __int128 m[4] = {0, 0, 0, 0};
    auto add = [&](int v) {
        const __int128 d = (long long)v - b;
        const __int128 d2 = d * d;
        m[0] += d; m[1] += d2; m[2] += d2 * d; m[3] += d2 * d2;
    };
    if (VEC) {
        const int4 *src = reinterpret_cast<const int4 *>(h) + (size_t)r * n4;
        for (uint32_t i = blockIdx.x * RED_THREADS + threadIdx.x; i < n4; i += gridDim.x * RED_THREADS) {
            const int4 q = __ldg(src + i);
            add(q.x); add(q.y); add(q.z); add(q.w);
        }
    } else {
        const int32_t *src = h + (size_t)r * n4;
        for (uint64_t i = (uint64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n4; i += (uint64_t)gridDim.x * RED_THREADS)
            add(__ldg(src + i));                           // 64-bit index, as in sums_kernel
    }
    for (int o = 16; o; o >>= 1)
#pragma unroll
        for (int k = 0; k < 4; ++k) m[k] += shfl_xor128(m[k], o);
    if ((threadIdx.x & 31) == 0)
#pragma unroll
        for (int k = 0; k < 4; ++k) add128(out + 8 * r + 2 * k, m[k]);
}

cudaError_t launch_moments(const int32_t *h, uint32_t L, uint32_t R, const long long *d_base,
                           unsigned long long *d_out, int sm_count, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(d_out, 0, (size_t)R * 8 * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    const bool vec = ((uint64_t)L * L) % 4 == 0;
    const uint64_t n4 = vec ? (uint64_t)L * L / 4 : (uint64_t)L * L;
    uint64_t bx = (n4 + RED_THREADS * 4 - 1) / (RED_THREADS * 4);
    const uint64_t want = ((uint64_t)(sm_count > 0 ? sm_count : 1) * 8 + R - 1) / R;
    if (bx > want) bx = want;
    if (bx < 1) bx = 1;
    for (uint32_t r0 = 0; r0 < R; r0 += 65535) {
        const uint32_t nr = R - r0 < 65535 ? R - r0 : 65535;
        if (vec) moments_kernel<true><<<dim3((unsigned)bx, nr), RED_THREADS, 0, st>>>(h + (size_t)r0 * L * L, (uint32_t)n4, d_base + r0,
                                                                                     d_out + 8 * (size_t)r0);
        else moments_kernel<false><<<dim3((unsigned)bx, nr), RED_THREADS, 0, st>>>(h + (size_t)r0 * L * L, (uint32_t)n4, d_base + r0,
                                                                                   d_out + 8 * (size_t)r0);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ---------------------------------------------------------------------------------------------
// Eq. (6) check of nr surfaces: counts the bonds (x, x+1) and (y, y+1), periodic, with
// |dh| > N into *d_bad.  Used by rsos_set_state: every engine relies on the invariant.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(RED_THREADS) violations_kernel(const int32_t *__restrict__ h, uint32_t L, uint32_t lgL,
                                                                 int32_t N, unsigned long long *d_bad)
{
    (void)lgL;
    const uint64_t n = (uint64_t)L * L;
    const int32_t *s = h + (size_t)blockIdx.y * n;
    unsigned int bad = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (uint64_t)gridDim.x * RED_THREADS) {
        const uint32_t y = (uint32_t)(i / L), x = (uint32_t)(i - (uint64_t)y * L);      // any L (D:2b)
        const int32_t c = s[i];
        const int32_t r = s[(size_t)y * L + (x + 1 == L ? 0 : x + 1)], d = s[(size_t)(y + 1 == L ? 0 : y + 1) * L + x];
        bad += (abs(c - r) > N) + (abs(c - d) > N);
    }
    for (int o = 16; o; o >>= 1) bad += __shfl_xor_sync(0xFFFFFFFFu, bad, o);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(d_bad, (unsigned long long)bad);
}

cudaError_t launch_violations(const int32_t *h, uint32_t L, uint32_t lgL, uint32_t nr, uint32_t N, unsigned long long *d_bad,
                              cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(d_bad, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    const uint64_t n = (uint64_t)L * L;
    const uint32_t bx = (uint32_t)((n + RED_THREADS * 8 - 1) / (RED_THREADS * 8) < 2048 ? (n + RED_THREADS * 8 - 1) / (RED_THREADS * 8) : 2048);
    for (uint32_t r0 = 0; r0 < nr; r0 += 65535) {
        const uint32_t cnt = nr - r0 < 65535 ? nr - r0 : 65535;
        violations_kernel<<<dim3(bx ? bx : 1, cnt), RED_THREADS, 0, st>>>(h + (size_t)r0 * n, L, lgL, (int32_t)N, d_bad);
    }
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// rsos_sums_static (include/rsos.h): the width sums for callers that must stay away from the CUDA
// allocator.  Same reduction as above (sums_kernel, Eq. 2), but the per-realization
// accumulators it adds into live in a fixed array that is part of the loaded library image
// instead of in a buffer some rsos_init obtained with cudaMalloc.
//
// g_static_red is a DEVICE object.  In host code its name only identifies the symbol; it is not an
// address a kernel can use.  static_scratch() asks the runtime for the real address once per
// device (cudaGetSymbolAddress, with that device current) and everything below works with that
// pointer.  One array per device, shared by every call and never cleared behind the caller's back:
// launch_sums zeroes the R rows it is going to use on the caller's stream before the kernel adds
// into them, and two calls whose work overlaps on the GPU (different streams, or two host threads)
// would add into the same rows -- the header says so.
// ---------------------------------------------------------------------------------------------
constexpr uint32_t STATIC_MAX_R = RSOS_STATIC_MAX_R;
constexpr int STATIC_MAX_DEVICES = 64;

static __device__ __align__(256) unsigned long long g_static_red[(size_t)STATIC_MAX_R * 4];   // 32 B per realization: 128 KiB

struct StaticScratch {
    bool ready = false;
    unsigned long long *ptr = nullptr;
    int sm_count = 0;
};
static StaticScratch g_static[STATIC_MAX_DEVICES];
static std::mutex g_static_mutex;

// The current device's copy of g_static_red and its SM count (looked up on the first call per device).
static cudaError_t static_scratch(unsigned long long **ptr, int *sm_count)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticScratch &s = g_static[dev];
    if (!s.ready) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_red);
        if (e != cudaSuccess) return e;
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        s.ptr = static_cast<unsigned long long *>(p);
        s.sm_count = sms;
        s.ready = true;
    }
    *ptr = s.ptr;
    *sm_count = s.sm_count;
    return cudaSuccess;
}

// Accumulator rows (S1, S2, max |h|, unused) -> the caller's three output arrays.
__global__ void __launch_bounds__(RED_THREADS) static_finish_kernel(const unsigned long long *__restrict__ red, uint32_t R,
                                                                    long long *S1, unsigned long long *S2, unsigned int *maxabs)
{
    const uint32_t r = blockIdx.x * RED_THREADS + threadIdx.x;
    if (r >= R) return;
    if (S1) S1[r] = (long long)red[4 * (size_t)r];
    if (S2) S2[r] = red[4 * (size_t)r + 1];
    if (maxabs) maxabs[r] = (unsigned int)red[4 * (size_t)r + 2];
}

cudaError_t launch_sums_static(const int32_t *h, uint32_t L, uint32_t R, long long *d_S1, unsigned long long *d_S2,
                               unsigned int *d_maxabs, cudaStream_t st)
{
    if (R < 1 || R > STATIC_MAX_R) return cudaErrorInvalidValue;          // rsos_sums_static reports this with a message first
    unsigned long long *red = nullptr;
    int sm_count = 0;
    cudaError_t e = static_scratch(&red, &sm_count);
    if (e != cudaSuccess) return e;
    e = launch_sums(h, L, R, red, sm_count, st);                          // clears rows 0..R-1 of red on st, then sums_kernel
    if (e != cudaSuccess) return e;
    static_finish_kernel<<<(R + RED_THREADS - 1) / RED_THREADS, RED_THREADS, 0, st>>>(red, R, d_S1, d_S2, d_maxabs);
    return cudaGetLastError();
}

}  // namespace rsos
