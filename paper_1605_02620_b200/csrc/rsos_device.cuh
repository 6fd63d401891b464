// rsos_device.cuh -- device-side building blocks shared by the update kernels of librsos.
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rsos {

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11), counter (c0..c3), key (k0,k1).  D:2 step 2.
// Written for the GPU: the two 32x32->64 products are IMAD.WIDE, the key schedule is folded into
// compile-time multiples of the Weyl constants so each round is 2 wide multiplies + 2 LOP3.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                uint32_t k0, uint32_t k1)
{
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    constexpr uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        const uint64_t p0 = (uint64_t)M0 * c0;
        const uint64_t p1 = (uint64_t)M1 * c2;
        const uint32_t ka = k0 + (uint32_t)i * W0;          // constant-folded offsets
        const uint32_t kb = k1 + (uint32_t)i * W1;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ ka;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ kb;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

// Everything a kernel needs to know about the run (passed by value).
struct Params {
    int32_t *h;                     // R * L * L heights, h[r][y][x]
    unsigned long long *accepted;   // R accepted-deposit counters
    uint32_t L, lgL;                // lattice side (power of two)
    uint32_t N;                     // Eq. (6) bound
    uint32_t R, first_real;
    uint32_t S, lgS, K;             // tile side, sub-sweeps per MCS (DT); S = L, K = 1 in RS mode
    uint32_t k0, k1;                // Philox key = (seed lo, seed hi)
    uint32_t *err;                  // device error word (bit flags), see ERR_*
    uint32_t *pk;                   // THREAD engine: packed working lattice, FB bits per site (rsos_pack.cu)
    uint32_t FB;                    // field bits of pk (2 or 4); 0 when there is no packed lattice
    uint32_t KL;                    // THREAD engine: lanes per tile (1, 2, 4 or 8)
    uint32_t poisson;               // 1: Poisson variant DTP(c) (D:2c): Poisson(4) attempts per cell and sub-sweep
    uint32_t multisurface;          // 1: shared-coordinate multisurface schedule MS (D:2d), MULTI engine
    uint32_t sm_count;              // SMs of the device (launch shapes)
    uint32_t general;               // 1: L is not a power of two -- general-L schedule RSG / DTG (D:2b), SIMPLE engine
    uint32_t T;                     // general DT mode: tiles per side, 2 * floor(L / 2S)
    uint32_t CS;                    // RESIDENT engine: thread blocks per cluster = per realization (1, 2, 4, 8 or 16)
};

enum : uint32_t {
    ERR_RECONSTRUCT = 1u,           // height reconstruction from differences did not divide exactly
};

// D:2 step 4: origin of sub-sweep u for realization rg: Philox counter (0, 0xFFFFFFFF, u, rg).
__device__ __forceinline__ void draw_origin(const Params &p, uint32_t u, uint32_t rg, uint32_t &ox, uint32_t &oy)
{
    const uint4 o = philox4x32_10(0u, 0xFFFFFFFFu, u, rg, p.k0, p.k1);
    ox = o.x & (p.L - 1);
    oy = o.y & (p.L - 1);
}

// ---------------------------------------------------------------------------------------------
// General-L schedule (D:2b): lattice sides that are not powers of two (P:79 L = 9605; P:204 irregular
// tilings).  Word stream of (tile id, u, r): word i = o[i & 3] of Philox(counter (i >> 2, tile id, u, r));
// draw(n): exactly uniform on [0, n) -- multiply-shift, a word whose low product half is below
// 2^32 mod n is rejected and the next word of the stream is taken.
// ---------------------------------------------------------------------------------------------
struct WordStream {
    uint32_t q, tile, u, rg, k0, k1, j;
    uint4 o;
    __device__ __forceinline__ WordStream(const Params &p, uint32_t tile_id, uint32_t u_, uint32_t rg_)
        : q(0), tile(tile_id), u(u_), rg(rg_), k0(p.k0), k1(p.k1), j(4), o(make_uint4(0, 0, 0, 0)) {}
    __device__ __forceinline__ uint32_t next()
    {
        if (j == 4) { o = philox4x32_10(q, tile, u, rg, k0, k1); ++q; j = 0; }
        const uint32_t v = j == 0 ? o.x : j == 1 ? o.y : j == 2 ? o.z : o.w;
        ++j;
        return v;
    }
    // thr = 2^32 mod n
    __device__ __forceinline__ uint32_t draw(uint32_t n, uint32_t thr)
    {
        for (;;) {
            const uint64_t m = (uint64_t)next() * n;
            if ((uint32_t)m >= thr) return (uint32_t)(m >> 32);
        }
    }
};

__device__ __forceinline__ uint32_t pow32_mod(uint32_t n) { return (uint32_t)(0x100000000ull % n); }
__device__ __forceinline__ uint32_t tile_edge(uint32_t i, uint32_t L, uint32_t T) { return (uint32_t)(((uint64_t)i * L) / T); }

}  // namespace rsos
