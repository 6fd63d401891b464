// Test-only helper: evaluates cuRAND's own Philox4x32-10 (the device header's host code path) so
// the oracle's Philox can be checked against an independent library routine (SURVEY 8c.3 pin P6).
// Never linked into the product library or the oracle.
// usage: curand_philox_host n seed   -> prints n lines "c0 c1 c2 c3 k0 k1 o0 o1 o2 o3" (hex)
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cuda_runtime.h>
#define QUALIFIERS static inline __host__ __device__
#include <curand_philox4x32_x.h>

static uint64_t sm64(uint64_t &s) {
    uint64_t z = (s += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

int main(int argc, char **argv) {
    long n = argc > 1 ? atol(argv[1]) : 16;
    uint64_t s = argc > 2 ? strtoull(argv[2], 0, 10) : 1;
    for (long i = 0; i < n; ++i) {
        uint64_t a = sm64(s), b = sm64(s), c = sm64(s);
        uint4 ctr = make_uint4((unsigned)a, (unsigned)(a >> 32), (unsigned)b, (unsigned)(b >> 32));
        uint2 key = make_uint2((unsigned)c, (unsigned)(c >> 32));
        if (i % 7 == 3) { ctr.y = 0xFFFFFFFFu; ctr.x = (unsigned)i; }   // the origin-draw counter shape
        uint4 o = curand_Philox4x32_10(ctr, key);
        printf("%08x %08x %08x %08x %08x %08x %08x %08x %08x %08x\n", ctr.x, ctr.y, ctr.z, ctr.w,
               key.x, key.y, o.x, o.y, o.z, o.w);
    }
    return 0;
}
