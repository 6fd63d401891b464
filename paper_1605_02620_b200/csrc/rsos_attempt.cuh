// rsos_attempt.cuh -- one deposition attempt on a tile window of packed sites in shared memory.
// Product code (CUDA path).  Shares nothing with oracle/.  Used by the lane-per-tile DT engine
// (rsos_thread.cu) and by the resident small-lattice engine (rsos_resident.cu).
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// Window format (D:4): a tile of S x S sites plus its one-site halo is (S + 2) rows of PW words; a
// site is FB bits, its height mod 2^FB (FB = 2 for N = 1, FB = 4 for N <= 7): under Eq. (6)
// nearest-neighbour differences lie in [-N, N] and are recoverable mod 2^FB.  Window
// column 0 is the left halo.  The windows of the NT = 32 / KL tiles a warp works on are stored
// word-interleaved: word w of tile g at smem[w * NT + g], so lanes of different tiles never share
// a bank.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

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

// ---------------------------------------------------------------------------------------------
// KL lanes share one tile (KL = 1, 2, 4 or 8; 32 / KL tiles per warp).  In every step the KL lanes of a
// group take KL consecutive attempts a0 + rank on the same snapshot of the tile.  A lane whose site
// is equal or adjacent to the site of a LOWER rank of its group, or shares a byte of packed sites
// with it, is "hazardous": it waits until the lower ranks have stored and then loads and decides
// again (rank by rank).  All other lanes cannot be affected by any lower rank, so their snapshot
// decision is the sequential one.  Stores are single bytes, so lanes that merely share a word do
// not interfere.  KL > 1 buys thread-level parallelism when a pass has few tiles (D:4).
// ---------------------------------------------------------------------------------------------
template <int LGS, int FB, int KL>
struct Attempt {
    using G = TGeom<LGS, FB>;
    static constexpr uint32_t NT = 32 / KL;               // tiles per warp = word stride (in words)
    static constexpr uint32_t WSB = NT * 4;               // byte stride between consecutive words of a tile
    static constexpr uint32_t ROWB = G::PW * WSB;         // byte stride between window rows
    uint32_t a0, ac;      // shared-memory byte addresses: word of the left neighbour, word of the site
    uint32_t sl, sc;      // bit positions of the left neighbour / the site inside those words
    uint32_t key;         // site code dy * S + dx = the low 2 lg S bits of the slot
    uint32_t w0, w1, wc, wu, wd;

    // v: 16-bit slot, dx = v & (S-1), dy = (v >> LGS) & (S-1)   (D:2 step 6)
    __device__ __forceinline__ void prep(uint32_t base, uint32_t v)
    {
        const uint32_t dx = v & (G::S - 1u), dy = (v >> LGS) & (G::S - 1u);
        const uint32_t bl = dx * FB, bc = bl + FB;        // window columns dx (left neighbour) and dx + 1 (site)
        const uint32_t row = base + (dy + 1u) * ROWB;
        a0 = row + (bl >> 5) * WSB;
        ac = row + (bc >> 5) * WSB;
        sl = bl & 31u;
        sc = bc & 31u;
        key = v & (G::S * G::S - 1u);
    }
    __device__ __forceinline__ void load()
    {
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(w0) : "r"(a0));
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(w1) : "r"(a0 + WSB));
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(wc) : "r"(ac));          // = w0 or w1; saves a select
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(wu) : "r"(ac - ROWB));
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(wd) : "r"(ac + ROWB));
    }
    // Eq. (6) test on the loaded words: rejected iff some neighbour sits at h - N, i.e.
    // nb == C - N mod 2^FB (D:3 (i)).  nw = the site's word with field C turned into C + 1 mod 2^FB.
    __device__ __forceinline__ bool decide(uint32_t N, uint32_t &nw) const
    {
        constexpr uint32_t M = G::M;
        const uint32_t t3 = __funnelshift_r(w0, w1, sl);           // fields: L, C, R (garbage above)
        // Everything is compared in the TOP FB bits of a register: a field is moved there by a multiply
        // with 2^(32 - FB - position) (IMAD: the fma pipe) instead of a shift (the alu pipe, which is
        // what this loop saturates first -- D:6).
        constexpr uint32_t TOP = M << (32 - FB), ONE = 1u << (32 - FB);
        const uint32_t m = ONE >> sc;                              // 2^(32 - FB - sc)
        auto mul = [](uint32_t a, uint32_t b) -> uint32_t {         // a real multiply: ptxas would turn a * 2^k into a shift
            uint32_t r;
            asm("mul.lo.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
            return r;
        };
        const uint32_t ct = mul(wc, m);                            // C on top
        const uint32_t tt = ct - N * ONE;                          // the blocking neighbour value C - N on top
        const uint32_t okL = ((t3 * ONE) ^ tt) & TOP;
        const uint32_t okR = ((t3 * (ONE >> (2 * FB))) ^ tt) & TOP;
        const uint32_t okU = (mul(wu, m) ^ tt) & TOP;
        const uint32_t okD = (mul(wd, m) ^ tt) & TOP;
        nw = wc ^ (((ct ^ (ct + ONE)) & TOP) >> (32 - FB - sc));   // field + 1 mod 2^FB
        return (okL != 0u) & (okR != 0u) & (okU != 0u) & (okD != 0u);
    }
    __device__ __forceinline__ void store(uint32_t nw) const
    {
        if (KL == 1) {
            asm volatile("st.shared.u32 [%0], %1;" :: "r"(ac), "r"(nw) : "memory");
        } else {                                           // only the byte holding the site
            asm volatile("st.shared.u8 [%0], %1;" :: "r"(ac + (sc >> 3)), "r"(nw >> (sc & 24u)) : "memory");
        }
    }
};

// Hazard between two attempts of one step, from their site codes alone (code = dy * S + dx).  Equal
// or adjacent sites have |d| in {0, 1, S}; sites in one byte of packed sites lie in one row within 3
// (2-bit) or 1 (4-bit) columns.  The test |d| <= 3 or |d| == S covers both and is conservative (it
// also fires across a row end): a false alarm only costs a reload.
template <int LGS>
__device__ __forceinline__ bool codes_clash(uint32_t a, uint32_t b)
{
    const uint32_t d = (uint32_t)abs((int32_t)(a - b));
    return (d <= 3u) | (d == (1u << LGS));
}

}  // namespace rsos
