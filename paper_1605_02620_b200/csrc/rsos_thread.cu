// rsos_thread.cu -- the LANE-PER-TILE update engine of the DT schedule (sm_100a).
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// One colour pass of one sub-sweep (D:2 steps 4-6; RSOS rule P:61-63 Eq. 6; double tiling with a
// moving origin P:77; independent realizations P:75).  A tile is owned by KL = 1, 2, 4 or 8 lanes of
// one warp (32 / KL tiles per warp) that run its S*S/K attempts in order, KL at a time; the result
// is the sequential one (one lane: by construction; more lanes: a lane whose site clashes with a
// lower rank's waits for it, see Attempt / group_finish).  What makes that fast (D:4, D:5):
//   * a site is FB bits, its height mod 2^FB (FB = 2 for N = 1, FB = 4 for N <= 7): under Eq. (6)
//     nearest-neighbour differences lie in [-N, N] and are recoverable mod 2^FB.  The working
//     lattice in HBM is packed the same way (rsos_pack.cu), so a tile window is (S+2) rows of
//     PW + 1 words instead of 4 bytes per site, and the int32 heights are rebuilt only on demand;
//   * the windows of a warp are stored word-interleaved, word w of tile g at smem[w * NT + g]
//     (NT = 32 / KL): lanes of different tiles never share a bank, and with one lane per tile every
//     shared-memory access of the attempt loop is conflict-free;
//   * window column 0 is the left halo (the packed row is funnel-shifted while staging), so the
//     attempt loop has no per-tile alignment term;
//   * fields are compared in the top bits of a register and moved there by multiplies, which run
//     on the fma pipe; the integer alu pipe is what the loop saturates first (D:6).
#include "rsos_attempt.cuh"
#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace rsos {

// Hazard of this lane's attempt against the lower ranks of its group (codes fetched by shuffles).
template <int LGS, int KL>
__device__ __forceinline__ bool group_hazard(uint32_t key, uint32_t rank)
{
    bool hz = false;
#pragma unroll
    for (int i = 1; i < KL; ++i) {
        const uint32_t ko = __shfl_up_sync(0xFFFFFFFFu, key, i);
        hz |= codes_clash<LGS>(key, ko) & ((uint32_t)i <= rank);
    }
    return hz;
}

// Second half of a step (KL > 1), after the loads of `a` were issued: decide on the snapshot,
// store unless hazardous, then let the hazardous lanes go rank by rank.  Returns 1 if accepted.
template <int LGS, int FB, int KL>
__device__ __forceinline__ uint32_t group_finish(Attempt<LGS, FB, KL> &a, bool hz, uint32_t N, uint32_t rank)
{
    constexpr uint32_t FULL = 0xFFFFFFFFu;
    uint32_t nw;
    bool ok = a.decide(N, nw);
    if (ok & !hz) a.store(nw);
    __syncwarp();
    uint32_t todo = __ballot_sync(FULL, hz);
    if (todo) {
        // ranks in ascending order; rank rr occupies the lanes rr, rr + KL, ... of the warp
#pragma unroll 1
        for (uint32_t rr = 1; rr < (uint32_t)KL && todo; ++rr) {
            uint32_t lanes_rr = 0;
#pragma unroll
            for (uint32_t g = 0; g < 32u / KL; ++g) lanes_rr |= 1u << (g * KL);
            lanes_rr <<= rr;
            if (todo & lanes_rr) {
                if (hz & (rank == rr)) {
                    a.load();
                    ok = a.decide(N, nw);
                    if (ok) a.store(nw);
                }
                __syncwarp();
                todo &= ~lanes_rr;
            }
        }
    }
    return ok ? 1u : 0u;
}

// Block b (one warp) runs tile set b: 32 / KL active tiles, KL lanes per tile.
template <int LGS, int FB, int KL>
__global__ void __launch_bounds__(32) thread_dt_kernel(Params p, uint32_t u, uint32_t colour)
{
    using G = TGeom<LGS, FB>;
    using At = Attempt<LGS, FB, KL>;
    constexpr uint32_t S = G::S, PW = G::PW, NTW = G::NTW, NT = At::NT;
    constexpr uint32_t FULL = 0xFFFFFFFFu;
    extern __shared__ __align__(16) uint32_t smem[];
    const uint32_t lane = threadIdx.x;
    const uint32_t grp = lane / KL, rank = lane % KL;
    const uint32_t L = p.L, Lm = L - 1;
    const uint32_t T = L >> LGS, half = T >> 1, ntile = half * half;
    const uint32_t total = p.R * ntile;
    uint32_t idx = blockIdx.x * NT + grp;
    const bool live = idx < total;
    if (!live) idx = total - 1u;                         // idle groups shadow the last tile, write nothing
    const uint32_t rl = idx / ntile, n = idx - rl * ntile;
    const uint32_t ti = n % half, tj = n / half;
    const uint32_t I = 2 * ti + (colour & 1u), J = 2 * tj + (colour >> 1);
    const uint32_t rg = p.first_real + rl;
    uint32_t ox, oy;
    draw_origin(p, u, rg, ox, oy);
    const uint32_t x0 = (ox + I * S) & Lm, y0 = (oy + J * S) & Lm;
    const uint32_t wpr = L >> G::LGSPW, wm = wpr - 1u;    // packed words per lattice row
    uint32_t *pk = p.pk + (size_t)rl * L * wpr;
    uint32_t *my = smem + grp;                            // word w of this group's tile: my[w * NT]
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(my);

    // ---- a3: stage rows y0-1 .. y0+S; window column X <-> lattice column x0 - 1 + X ------------
    {
        const uint32_t gxs = (x0 - 1u) & Lm;
        const uint32_t ws = gxs >> G::LGSPW, o = (gxs & (G::SPW - 1u)) * FB;
#pragma unroll 2
        for (uint32_t yr = rank; yr < G::ROWS; yr += KL) {
            const uint32_t *rowp = pk + (size_t)((y0 - 1u + yr) & Lm) * wpr;
            uint32_t g[PW + 1];
#pragma unroll
            for (uint32_t k = 0; k <= PW; ++k) g[k] = rowp[(ws + k) & wm];
#pragma unroll
            for (uint32_t k = 0; k < PW; ++k) my[(yr * PW + k) * NT] = __funnelshift_r(g[k], g[k + 1], o);
        }
    }
    __syncwarp();

    // ---- a1 + a4: A attempts in order, KL per step.  Attempt a takes the 16-bit slot a & 7 of
    // Philox call a >> 3 (D:2 step 6).  A batch is KL calls = 8 steps; rank r computes call
    // batch * KL + r and the slots travel inside the group by shuffles.
    const uint32_t A = (S * S) / p.K;
    const uint32_t tile_id = J * T + I;
    const uint32_t N = p.N;
    uint32_t nacc = 0;
    if (KL == 1) {
#pragma unroll 1
        for (uint32_t q = 0; q < A / 8u; ++q) {
            const uint4 o = philox4x32_10(q, tile_id, u, rg, p.k0, p.k1);
            const uint32_t ow[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
            for (uint32_t w = 0; w < 8; ++w) {
                At a;
                a.prep(base, (ow[w >> 1] >> (16u * (w & 1u))) & 0xFFFFu);
                a.load();
                uint32_t nw;
                const bool ok = a.decide(N, nw);
                if (ok) a.store(nw);
                nacc += ok ? 1u : 0u;
            }
        }
    } else {
        // KL lanes per tile.  The slot shuffles, the address arithmetic and the hazard test of step
        // w + 1 depend on nothing in memory; they are issued right after the loads of step w so that
        // they fill its latency instead of lengthening the chain load -> decide -> store -> vote.
        const uint32_t nbatch = A / (8u * KL);
        uint4 o = philox4x32_10(rank, tile_id, u, rg, p.k0, p.k1);
        // slot of step w of the batch whose calls are in (o of every rank): attempt KL*w + rank
        auto slot_of = [&](const uint4 &c, uint32_t w) -> uint32_t {
            const uint32_t cw[4] = {c.x, c.y, c.z, c.w};
            if (KL == 2) {                                // call w >> 2, slot 2(w & 3) + rank
                const uint32_t x = __shfl_sync(FULL, cw[w & 3u], grp * KL + (w >> 2));
                return rank ? x >> 16 : x & 0xFFFFu;
            } else if (KL == 4) {                         // call w >> 1, slot 4(w & 1) + rank
                const uint32_t src = grp * KL + (w >> 1);
                const uint32_t xa = __shfl_sync(FULL, cw[2u * (w & 1u)], src);
                const uint32_t xb = __shfl_sync(FULL, cw[2u * (w & 1u) + 1u], src);
                const uint32_t x = (rank & 2u) ? xb : xa;
                return (rank & 1u) ? x >> 16 : x & 0xFFFFu;
            } else {                                      // KL == 8: call w, slot rank
                const uint32_t src = grp * KL + w;
                const uint32_t x0 = __shfl_sync(FULL, cw[0], src), x1 = __shfl_sync(FULL, cw[1], src);
                const uint32_t x2 = __shfl_sync(FULL, cw[2], src), x3 = __shfl_sync(FULL, cw[3], src);
                const uint32_t x = (rank & 4u) ? ((rank & 2u) ? x3 : x2) : ((rank & 2u) ? x1 : x0);
                return (rank & 1u) ? x >> 16 : x & 0xFFFFu;
            }
        };
        if (KL == 2) {
            // Two lanes per tile: the pair swaps its two Philox calls once per batch (4 shuffles), so
            // both lanes hold calls 2b and 2b + 1.  Step w takes word w of the 8: rank 0 the low half
            // (attempt 2w), rank 1 the high half (attempt 2w + 1) -- each lane sees its partner's slot
            // in the same register and needs no shuffle for the hazard test.
            auto swap4 = [&](const uint4 &c) -> uint4 {
                return make_uint4(__shfl_xor_sync(FULL, c.x, 1), __shfl_xor_sync(FULL, c.y, 1),
                                  __shfl_xor_sync(FULL, c.z, 1), __shfl_xor_sync(FULL, c.w, 1));
            };
            constexpr uint32_t CM = S * S - 1u;
            auto mine = [&](uint32_t x) -> uint32_t { return rank ? x >> 16 : x & 0xFFFFu; };
            auto clash = [&](uint32_t x) -> bool { return (rank != 0u) & codes_clash<LGS>((x >> 16) & CM, x & CM); };
            uint4 po = swap4(o);
            uint32_t c[9];
            c[0] = rank ? po.x : o.x; c[1] = rank ? po.y : o.y; c[2] = rank ? po.z : o.z; c[3] = rank ? po.w : o.w;
            c[4] = rank ? o.x : po.x; c[5] = rank ? o.y : po.y; c[6] = rank ? o.z : po.z; c[7] = rank ? o.w : po.w;
            At cur;
            cur.prep(base, mine(c[0]));
            bool hz = clash(c[0]);
#pragma unroll 1
            for (uint32_t batch = 0; batch < nbatch; ++batch) {
                const uint4 on = philox4x32_10((batch + 1u) * KL + rank, tile_id, u, rg, p.k0, p.k1);   // last one unused
                const uint4 pon = swap4(on);
                c[8] = rank ? pon.x : on.x;
#pragma unroll
                for (uint32_t w = 0; w < 8; ++w) {
                    cur.load();
                    At nxt;
                    nxt.prep(base, mine(c[w + 1u]));
                    const bool hzn = clash(c[w + 1u]);
                    nacc += group_finish<LGS, FB, KL>(cur, hz, N, rank);
                    cur = nxt;
                    hz = hzn;
                }
                c[0] = c[8]; c[1] = rank ? pon.y : on.y; c[2] = rank ? pon.z : on.z; c[3] = rank ? pon.w : on.w;
                c[4] = rank ? on.x : pon.x; c[5] = rank ? on.y : pon.y; c[6] = rank ? on.z : pon.z; c[7] = rank ? on.w : pon.w;
            }
        } else {
        At cur;
        cur.prep(base, slot_of(o, 0u));
        bool hz = group_hazard<LGS, KL>(cur.key, rank);
#pragma unroll 1
        for (uint32_t batch = 0; batch < nbatch; ++batch) {
            const uint4 on = philox4x32_10((batch + 1u) * KL + rank, tile_id, u, rg, p.k0, p.k1);   // last one unused
#pragma unroll
            for (uint32_t w = 0; w < 8; ++w) {
                cur.load();
                At nxt;
                nxt.prep(base, w < 7u ? slot_of(o, w + 1u) : slot_of(on, 0u));
                const bool hzn = group_hazard<LGS, KL>(nxt.key, rank);
                nacc += group_finish<LGS, FB, KL>(cur, hz, N, rank);
                cur = nxt;
                hz = hzn;
            }
            o = on;
        }
        }
    }
    __syncwarp();

    // ---- a5: write back the S x S tile bits.  A tile row is TBITS bits starting at bit ob of
    // packed word wsb; whole words are stored, the (at most two) partial edge words are merged
    // with the lattice word.  No other tile of this pass touches those words: tiles of one colour
    // are S >= SPW sites apart (D:5).
    if (live) {
        const uint32_t wsb = x0 >> G::LGSPW, ob = (x0 & (G::SPW - 1u)) * FB;
#pragma unroll 1
        for (uint32_t Y = 1u + rank; Y <= S; Y += KL) {
            uint32_t *rowp = pk + (size_t)((y0 - 1u + Y) & Lm) * wpr;
            uint32_t w[PW + 1];
#pragma unroll
            for (uint32_t k = 0; k < PW; ++k) w[k] = my[(Y * PW + k) * NT];
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
                else if (mk != 0u) {                        // partial word: clear my bits, then set them (no
                    atomicAnd(dst, ~mk);                    // load to wait for; nobody else writes this word
                    atomicOr(dst, gk);                      // in this pass and nobody reads my bits)
                }
            }
        }
        if (nacc) atomicAdd(p.accepted + rl, (unsigned long long)nacc);
    }
}

// =============================================================================================
// Host-side launchers
// =============================================================================================
template <int LGS, int FB, int KL>
static cudaError_t thread_dt_t(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st, int what,
                               size_t *out)
{
    const size_t sm = (size_t)(32 / KL) * TGeom<LGS, FB>::WORDS * 4;
    if (what == 0) { *out = sm; return cudaSuccess; }
    if (what == 1)
        return cudaFuncSetAttribute(thread_dt_kernel<LGS, FB, KL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    thread_dt_kernel<LGS, FB, KL><<<blocks, 32, sm, st>>>(p, u, colour);
    return cudaGetLastError();
}

template <int LGS, int FB>
static cudaError_t thread_dt_k(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st, int what,
                               size_t *out)
{
    switch (p.KL) {
        case 1: return thread_dt_t<LGS, FB, 1>(p, u, colour, blocks, st, what, out);
        case 2: return thread_dt_t<LGS, FB, 2>(p, u, colour, blocks, st, what, out);
        case 4: return thread_dt_t<LGS, FB, 4>(p, u, colour, blocks, st, what, out);
        case 8: return thread_dt_t<LGS, FB, 8>(p, u, colour, blocks, st, what, out);
        default: return cudaErrorInvalidValue;
    }
}

static cudaError_t thread_dispatch(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st,
                                   int what, size_t *out)
{
    const bool two = p.FB == 2;
    switch (p.lgS) {
        case 3: return thread_dt_k<3, 4>(p, u, colour, blocks, st, what, out);      // S = 8 < 16 sites per 2-bit word
        case 4: return two ? thread_dt_k<4, 2>(p, u, colour, blocks, st, what, out)
                           : thread_dt_k<4, 4>(p, u, colour, blocks, st, what, out);
        case 5: return two ? thread_dt_k<5, 2>(p, u, colour, blocks, st, what, out)
                           : thread_dt_k<5, 4>(p, u, colour, blocks, st, what, out);
        case 6: return two ? thread_dt_k<6, 2>(p, u, colour, blocks, st, what, out)
                           : thread_dt_k<6, 4>(p, u, colour, blocks, st, what, out);
        default: return cudaErrorInvalidValue;
    }
}

// Field width of the packed lattice (D:5): 2 bits when N = 1 and a tile is at least one 2-bit
// word wide (so that tiles of one colour never share a packed word), else 4 bits (N <= 7).
uint32_t thread_dt_field_bits(uint32_t N, uint32_t S) { return (N <= 1u && S >= 16u) ? 2u : 4u; }

// Lanes per tile (D:4): 2 when a colour pass then has about six warps per SM, else 4.  More lanes per
// tile cost instructions (shuffles, hazard test, votes) and buy resident warps: a tile window is
// 1.3 KB of shared memory whoever works on it.  Measured on B200 (G attempts/s at 1 / 2 / 4 / 8
// lanes): C4, 65536 tiles per pass: 284 / 292 / 253 / -; C3, 16384: 233 / 257 / 209 / -;
// C2, 8192: 110 / 142 / 195 / 143.
// With 4-bit sites a window is twice as large (half the resident warps): 4 lanes (C3 at N = 2..4:
// 112 / 156 / 174 G attempts/s at 1 / 2 / 4 lanes).
uint32_t thread_dt_lanes_per_tile(uint64_t pass_tiles, int sm_count, uint32_t field_bits)
{
    if (field_bits > 2) return 4u;
    return pass_tiles * 2 / 32 >= (uint64_t)sm_count * 6 ? 2u : 4u;
}

size_t thread_dt_smem(const Params &p)
{
    if (p.general) return gthread_smem(p);
    size_t sm = 0;
    thread_dispatch(p, 0, 0, 0, nullptr, 0, &sm);
    return sm;
}

cudaError_t thread_dt_configure(const Params &p)
{
    return p.general ? gthread_configure(p) : thread_dispatch(p, 0, 0, 0, nullptr, 1, nullptr);
}

uint32_t thread_dt_blocks(const Params &p)
{
    if (p.general) return gthread_blocks(p);
    const uint32_t T = p.L >> p.lgS, half = T >> 1;
    const uint64_t tiles = (uint64_t)p.R * half * half;
    const uint32_t nt = 32u / p.KL;
    return (uint32_t)((tiles + nt - 1) / nt);
}

cudaError_t thread_dt_launch(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st)
{
    if (p.general) return gthread_launch(p, u, colour, st);     // lattice side not a power of two: rsos_gthread.cu
    return thread_dispatch(p, u, colour, blocks, st, 2, nullptr);
}

}  // namespace rsos
