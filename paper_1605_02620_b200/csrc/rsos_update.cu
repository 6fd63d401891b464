// rsos_update.cu -- the RSOS update kernels (sm_100a).  Product code; shares nothing with oracle/.
//
// Citations: P:n = PAPER.md line n; D:x = DESIGN.md section x.
//
// Three of the four engines (the lane-per-tile THREAD engine lives in rsos_thread.cu), all executing the seeded schedule of D:2 (RSOS rule P:61-63 Eq. 6, double tiling
// with a moving origin P:77, independent realizations P:75) and producing identical heights:
//
//   simple_*   one THREAD per active tile, heights in global memory, the literal loop nest.
//   warp_dt    one WARP per active tile.  The (S+2)^2 window is staged into shared memory as
//              6-bit heights (mod 64) in 2x2-site blocks per 32-bit word, 32 consecutive attempts
//              are evaluated at once and committed as the longest conflict-free prefix, so the
//              result equals the sequential one exactly (D:4).
//   warp_rs    RS mode: one warp per realization, the whole periodic lattice stays in shared
//              memory for all MCS of the call (D:4, "on-chip").
#include "rsos_device.cuh"
#include "rsos_internal.h"

namespace rsos {

// =============================================================================================
// SIMPLE engine: the literal loop nest of D:2 step 6, one thread per tile.
// =============================================================================================
__device__ __forceinline__ uint32_t simple_run_tile(const Params &p, int32_t *h, uint32_t rg, uint32_t u,
                                                    uint32_t tile_id, uint32_t x0, uint32_t y0,
                                                    uint32_t Se, uint32_t lgSe, uint64_t A)
{
    const uint32_t L = p.L, Lm = L - 1;
    const uint32_t w16 = (2 * lgSe <= 16);
    const uint32_t lg_ns = w16 ? 3 : 2;
    const int32_t N = (int32_t)p.N;
    uint32_t nacc = 0;
    uint4 o = make_uint4(0, 0, 0, 0);
    uint32_t have_q = 0xFFFFFFFFu;
    for (uint64_t a = 0; a < A; ++a) {
        const uint32_t q = (uint32_t)(a >> lg_ns);                  // D:2 step 6: call a / ns, slot a % ns
        const uint32_t j = (uint32_t)a & ((1u << lg_ns) - 1u);
        if (q != have_q) { o = philox4x32_10(q, tile_id, u, rg, p.k0, p.k1); have_q = q; }
        uint32_t v;
        if (w16) {
            const uint32_t word = (j >> 1) == 0 ? o.x : (j >> 1) == 1 ? o.y : (j >> 1) == 2 ? o.z : o.w;
            v = (word >> (16u * (j & 1u))) & 0xFFFFu;
        } else {
            v = j == 0 ? o.x : j == 1 ? o.y : j == 2 ? o.z : o.w;
        }
        const uint32_t dx = v & (Se - 1), dy = (v >> lgSe) & (Se - 1);
        const uint32_t x = (x0 + dx) & Lm, y = (y0 + dy) & Lm;
        int32_t *row = h + (size_t)y * L;
        const int32_t c = row[x] + 1;
        const int32_t l = row[(x - 1) & Lm], r = row[(x + 1) & Lm];
        const int32_t up = h[(size_t)((y - 1) & Lm) * L + x], dn = h[(size_t)((y + 1) & Lm) * L + x];
        const bool ok = abs(c - l) <= N && abs(c - r) <= N && abs(c - up) <= N && abs(c - dn) <= N;
        if (ok) { row[x] = c; ++nacc; }
    }
    return nacc;
}

// General-L form (D:2b): a tile of w x hgt sites whose first site is (x0, y0); A attempts, each
// s = draw(w * hgt), dx = s mod w, dy = s div w, site ((x0 + dx) mod L, (y0 + dy) mod L).
__device__ __forceinline__ uint32_t general_run_tile(const Params &p, int32_t *h, uint32_t rg, uint32_t u, uint32_t tile_id,
                                                     uint32_t x0, uint32_t y0, uint32_t w, uint32_t hgt, uint64_t A)
{
    const uint32_t L = p.L, n = w * hgt, thr = pow32_mod(n);
    const int32_t N = (int32_t)p.N;
    WordStream ws(p, tile_id, u, rg);
    uint32_t nacc = 0;
    for (uint64_t a = 0; a < A; ++a) {
        const uint32_t s = ws.draw(n, thr);
        const uint32_t dy = s / w, dx = s - dy * w;
        uint32_t x = x0 + dx, y = y0 + dy;
        if (x >= L) x -= L;
        if (y >= L) y -= L;
        const uint32_t xm = x ? x - 1 : L - 1, xp = x + 1 == L ? 0 : x + 1;
        const uint32_t ym = y ? y - 1 : L - 1, yp = y + 1 == L ? 0 : y + 1;
        int32_t *row = h + (size_t)y * L;
        const int32_t c = row[x] + 1;
        const int32_t l = row[xm], r = row[xp];
        const int32_t up = h[(size_t)ym * L + x], dn = h[(size_t)yp * L + x];
        const bool ok = abs(c - l) <= N && abs(c - r) <= N && abs(c - up) <= N && abs(c - dn) <= N;
        if (ok) { row[x] = c; ++nacc; }
    }
    return nacc;
}

// One colour pass of the general-L DT schedule: T = 2 floor(L / 2S) tiles per side with edges floor(i L / T); the
// origin of sub-sweep u comes from the stream of tile id 0xFFFFFFFF; in sub-sweep k = u mod K a tile of n sites makes
// floor((k + 1) n / K) - floor(k n / K) attempts (n per MCS).
__device__ __forceinline__ void general_dt_pass(const Params &p, uint32_t u, uint32_t colour, uint32_t idx)
{
    const uint32_t L = p.L, T = p.T, half = T >> 1, ntile = half * half;
    if (idx >= p.R * ntile) return;
    const uint32_t rl = idx / ntile, n = idx - rl * ntile;
    const uint32_t I = 2 * (n % half) + (colour & 1u), J = 2 * (n / half) + (colour >> 1);
    const uint32_t rg = p.first_real + rl;
    WordStream os(p, 0xFFFFFFFFu, u, rg);
    const uint32_t thrL = pow32_mod(L);
    const uint32_t ox = os.draw(L, thrL);
    const uint32_t oy = os.draw(L, thrL);
    const uint32_t bx = tile_edge(I, L, T), by = tile_edge(J, L, T);
    const uint32_t w = tile_edge(I + 1, L, T) - bx, hgt = tile_edge(J + 1, L, T) - by;
    const uint64_t sites = (uint64_t)w * hgt, k = u & (p.K - 1u);
    const uint64_t A = ((k + 1) * sites) / p.K - (k * sites) / p.K;
    int32_t *h = p.h + (size_t)rl * L * L;
    const uint32_t nacc = general_run_tile(p, h, rg, u, J * T + I, (ox + bx) % L, (oy + by) % L, w, hgt, A);
    if (nacc) atomicAdd(p.accepted + rl, (unsigned long long)nacc);
}

// ---------------------------------------------------------------------------------------------
// General-L DT pass with tile windows in shared memory (D:2b, N <= 7).  A warp owns GW_NT = 16 tiles: the 32 lanes
// stage the (w + 2) x (hgt + 2) windows one tile after the other (coalesced int32 rows -> one byte per site, the
// height mod 256), lane g < 16 then runs the attempts of tile g in order on its window, and the warp writes the
// interiors back as h += (new byte - old byte) mod 256.  Word j of tile g lives at smem[j * 16 + g], so the 16
// working lanes never share a bank.  Exact: Eq. (6) needs only differences (|dh| <= N < 128 survives mod 256), and
// for N <= 7 no site can gain 256 within one pass (raising one site by 256 forces >= 256 + 4*242 + 8*228 + ... more
// than the (2S)^2 attempts a tile has), so the byte delta is the true one.
// ---------------------------------------------------------------------------------------------
constexpr uint32_t GW_NT = 16;
constexpr uint32_t GW_MAX_COLS = 128;      // staging and write-back move 4 chunks of 32 lanes per window row: columns 0..127

__global__ void __launch_bounds__(32) general_window_kernel(Params p, uint32_t u, uint32_t colour, uint32_t pww, uint32_t nrows)
{
    extern __shared__ __align__(16) uint32_t gsm[];
    uint8_t *win = reinterpret_cast<uint8_t *>(gsm);
    const uint32_t lane = threadIdx.x;
    const uint32_t L = p.L, T = p.T, half = T >> 1, ntile = half * half;
    const uint32_t total = p.R * ntile;
    const uint32_t thrL = pow32_mod(L);
    (void)nrows;

    // geometry of tile slot g of this warp (uniform over the lanes that ask for the same g)
    struct Tile { uint32_t rl, x0, y0, w, hgt, id, rg; bool live; };
    auto tile_of = [&](uint32_t g) -> Tile {
        Tile t;
        const uint32_t idx = blockIdx.x * GW_NT + g;
        t.live = idx < total;
        const uint32_t i = t.live ? idx : 0u;
        t.rl = i / ntile;
        const uint32_t n = i - t.rl * ntile;
        const uint32_t I = 2 * (n % half) + (colour & 1u), J = 2 * (n / half) + (colour >> 1);
        t.rg = p.first_real + t.rl;
        WordStream os(p, 0xFFFFFFFFu, u, t.rg);
        const uint32_t ox = os.draw(L, thrL);
        const uint32_t oy = os.draw(L, thrL);
        const uint32_t bx = tile_edge(I, L, T), by = tile_edge(J, L, T);
        t.w = tile_edge(I + 1, L, T) - bx;
        t.hgt = tile_edge(J + 1, L, T) - by;
        t.x0 = (ox + bx) % L;
        t.y0 = (oy + by) % L;
        t.id = J * T + I;
        return t;
    };
    // byte address of window site (col, row) of tile g; col, row = 0 is the halo
    auto waddr = [&](uint32_t g, uint32_t col, uint32_t row) -> uint32_t {
        return (((row * pww + (col >> 2)) * GW_NT + g) << 2) + (col & 3u);
    };

    // ---- a3: stage.  Four rows x up to four column chunks of loads are issued before the first byte is stored, so a
    // dozen global loads are in flight per lane (a lone warp hides no latency otherwise).
    auto wrap3 = [&](uint32_t v) -> uint32_t { return v - ((v >= 2u * L) ? 2u * L : (v >= L ? L : 0u)); };
    for (uint32_t g = 0; g < GW_NT; ++g) {
        const Tile t = tile_of(g);
        if (!t.live) break;                                              // tiles are assigned in order: the rest is idle too
        const int32_t *h = p.h + (size_t)t.rl * L * L;
        const uint32_t ncol = t.w + 2u, nrow = t.hgt + 2u;
        for (uint32_t row0 = 0; row0 < nrow; row0 += 4u) {
            int32_t v[4][4];
#pragma unroll
            for (uint32_t dr = 0; dr < 4; ++dr) {
                const uint32_t row = row0 + dr < nrow ? row0 + dr : nrow - 1u;
                const int32_t *src = h + (size_t)wrap3(t.y0 + L - 1u + row) * L;
#pragma unroll
                for (uint32_t dc = 0; dc < 4; ++dc) {
                    const uint32_t col = lane + 32u * dc;
                    v[dr][dc] = col < ncol ? src[wrap3(t.x0 + L - 1u + col)] : 0;
                }
            }
#pragma unroll
            for (uint32_t dr = 0; dr < 4; ++dr)
#pragma unroll
                for (uint32_t dc = 0; dc < 4; ++dc) {
                    const uint32_t col = lane + 32u * dc;
                    if (row0 + dr < nrow && col < ncol) win[waddr(g, col, row0 + dr)] = (uint8_t)((uint32_t)v[dr][dc] & 0xFFu);
                }
        }
    }
    __syncwarp();

    // ---- a1 + a4: lane g runs tile g ----------------------------------------------------------------------------------
    uint32_t nacc = 0;
    Tile me = tile_of(lane < GW_NT ? lane : 0u);
    if (lane < GW_NT && me.live) {
        const uint32_t n = me.w * me.hgt, thr = pow32_mod(n);
        const uint64_t k = u & (p.K - 1u);
        const uint64_t A = ((k + 1) * (uint64_t)n) / p.K - (k * (uint64_t)n) / p.K;
        const int32_t N = (int32_t)p.N;
        WordStream ws(p, me.id, u, me.rg);
        const uint32_t inv_w = 0xFFFFFFFFu / me.w;                      // s / w = mulhi(s, inv_w) or one more (s < 2^15)
        for (uint64_t a = 0; a < A; ++a) {
            const uint32_t s = ws.draw(n, thr);
            uint32_t dy = __umulhi(s, inv_w);
            uint32_t dx = s - dy * me.w;
            if (dx >= me.w) { dx -= me.w; ++dy; }
            const uint32_t aC = waddr(lane, dx + 1u, dy + 1u);
            const uint32_t c = (uint32_t)win[aC] + 1u;
            const uint32_t l = win[waddr(lane, dx, dy + 1u)], r = win[waddr(lane, dx + 2u, dy + 1u)];
            const uint32_t up = win[aC - pww * GW_NT * 4u], dn = win[aC + pww * GW_NT * 4u];
            auto far = [&](uint32_t nb) -> bool { return abs((int32_t)(int8_t)((c - nb) & 0xFFu)) > N; };
            if (!(far(l) | far(r) | far(up) | far(dn))) { win[aC] = (uint8_t)c; ++nacc; }
        }
    }
    __syncwarp();

    // ---- a5: write back the interiors (same blocking: 4 rows x 4 column chunks of loads in flight) --------------------------
    for (uint32_t g = 0; g < GW_NT; ++g) {
        const Tile t = tile_of(g);
        if (!t.live) break;
        int32_t *h = p.h + (size_t)t.rl * L * L;
        for (uint32_t row0 = 1; row0 <= t.hgt; row0 += 4u) {
            int32_t old[4][4];
            int32_t *dst[4][4];
#pragma unroll
            for (uint32_t dr = 0; dr < 4; ++dr) {
                const uint32_t row = row0 + dr <= t.hgt ? row0 + dr : t.hgt;
                int32_t *rowp = h + (size_t)wrap3(t.y0 + row - 1u) * L;
#pragma unroll
                for (uint32_t dc = 0; dc < 4; ++dc) {
                    const uint32_t col = 1u + lane + 32u * dc;
                    dst[dr][dc] = rowp + wrap3(t.x0 + (col <= t.w ? col : 1u) - 1u);
                    old[dr][dc] = (row0 + dr <= t.hgt && col <= t.w) ? *dst[dr][dc] : 0;
                }
            }
#pragma unroll
            for (uint32_t dr = 0; dr < 4; ++dr)
#pragma unroll
                for (uint32_t dc = 0; dc < 4; ++dc) {
                    const uint32_t col = 1u + lane + 32u * dc;
                    if (row0 + dr <= t.hgt && col <= t.w) {
                        const uint32_t d = ((uint32_t)win[waddr(g, col, row0 + dr)] - (uint32_t)old[dr][dc]) & 0xFFu;
                        if (d) *dst[dr][dc] = old[dr][dc] + (int32_t)d;
                    }
                }
        }
    }
    if (lane < GW_NT && me.live && nacc) atomicAdd(p.accepted + me.rl, (unsigned long long)nacc);
}

// window geometry of the general-L pass: words per window row and rows; 0 if the windows of 16 tiles do not fit
static bool general_window_shape(const Params &p, uint32_t *pww, uint32_t *nrows, size_t *smem)
{
    if (!p.general || !p.T || p.N > 7) return false;
    const uint32_t wmax = (p.L + p.T - 1) / p.T;                       // ceil(L / T): the larger of the two tile sizes
    if (wmax + 2 > GW_MAX_COLS) return false;                          // wider windows: simple_dt_kernel (the shared-memory
                                                                       // cap below is tighter today; this keeps it explicit)
    *pww = (wmax + 2 + 3) / 4;
    *nrows = wmax + 2;
    *smem = (size_t)*pww * *nrows * GW_NT * 4;
    return *smem <= 200u * 1024u;
}

__global__ void __launch_bounds__(128) simple_dt_kernel(Params p, uint32_t u, uint32_t colour)
{
    if (p.general) { general_dt_pass(p, u, colour, blockIdx.x * blockDim.x + threadIdx.x); return; }
    const uint32_t T = p.L >> p.lgS, half = T >> 1, ntile = half * half;
    const uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= p.R * ntile) return;
    const uint32_t rl = idx / ntile, n = idx - rl * ntile;
    const uint32_t i = n % half, j = n / half;
    const uint32_t I = 2 * i + (colour & 1u), J = 2 * j + (colour >> 1);
    const uint32_t rg = p.first_real + rl;
    uint32_t ox, oy;
    draw_origin(p, u, rg, ox, oy);
    const uint32_t x0 = (ox + I * p.S) & (p.L - 1), y0 = (oy + J * p.S) & (p.L - 1);
    int32_t *h = p.h + (size_t)rl * p.L * p.L;
    const uint32_t nacc = simple_run_tile(p, h, rg, u, J * T + I, x0, y0, p.S, p.lgS, ((uint64_t)p.S * p.S) / p.K);
    if (nacc) atomicAdd(p.accepted + rl, (unsigned long long)nacc);
}

__global__ void __launch_bounds__(32) simple_rs_kernel(Params p, uint32_t t0, uint32_t mcs)
{
    const uint32_t rl = blockIdx.x * blockDim.x + threadIdx.x;
    if (rl >= p.R) return;
    int32_t *h = p.h + (size_t)rl * p.L * p.L;
    unsigned long long nacc = 0;
    for (uint32_t m = 0; m < mcs; ++m)
        nacc += p.general ? general_run_tile(p, h, p.first_real + rl, t0 + m, 0u, 0u, 0u, p.L, p.L, (uint64_t)p.L * p.L)
                          : simple_run_tile(p, h, p.first_real + rl, t0 + m, 0u, 0u, 0u, p.L, p.lgL, (uint64_t)p.L * p.L);
    if (nacc) atomicAdd(p.accepted + rl, nacc);
}

// =============================================================================================
// WARP engines.  On-chip format (D:4): heights mod 64 (N <= 31 makes every nearest-neighbour
// difference recoverable), four sites of a 2x2 block per 32-bit word, byte k = (Y&1)*2 + (X&1),
// low 6 bits = height, top 2 bits of the four bytes = the id of the lane that last wrote the word.
// =============================================================================================
constexpr uint32_t HMASK = 0x3F3F3F3Fu;

__device__ __forceinline__ uint32_t lane_tag(uint32_t lane)
{
    return ((lane & 3u) << 6) | (((lane >> 2) & 3u) << 14) | (((lane >> 4) & 1u) << 22);
}

// Geometry of the shared-memory window of one warp.
//   DT  : window of (S+8) x (S+4) sites whose origin (xa, ya) is 4-/2-aligned in GLOBAL lattice
//         coordinates; it contains the S x S tile at (offx, offy) and its 1-site halo.
//   RS  : the whole L x L lattice, periodic.
template <int LGS, bool WRAP>
struct Geom {
    static constexpr uint32_t S = 1u << LGS;
    static constexpr uint32_t PITCH = WRAP ? (S / 2) : (S + 8) / 2;        // words per block row
    static constexpr uint32_t ROWS = WRAP ? (S / 2) : (S + 4) / 2;         // block rows
    static constexpr uint32_t WORDS = PITCH * ROWS;
    static constexpr uint32_t NBM = S / 2 - 1;                             // block-index mask (RS)
};

// ---------------------------------------------------------------------------------------------
// All A attempts of one tile by one warp, exactly as if executed one after another (D:2 step 6).
//
// 32 consecutive attempts a0 .. a0+31 are in flight, attempt a on lane a & 31.  Attempt a takes the
// 16-bit slot a & 7 of Philox call a >> 3 (D:2 step 6, reading Q16); lane l computes the calls
// 32 g + l of every group g of 256 attempts and the slots reach their attempts through shuffles.
// Window step (D:4):
//   R  every lane reads the three words holding its 5-point stencil;
//   D  decides on that snapshot: under Eq. (6) the deposit is rejected iff some neighbour
//      equals h - N (mod 64);
//   W  accepting lanes store the updated word, tagged with their lane id;
//   V  every lane re-reads its three words.  A lane is DIRTY if a stencil site changed under it or
//      its own store is not what the word now holds -- i.e. another accepting lane of this window
//      wrote the same or an adjacent site (or the same word).
//   C  f = lowest dirty rank (rank = position in the window); ranks < f are final.  Lanes >= f
//      whose store survived undo it; all of them are retried in the next window, which starts at
//      a0 + f.  Rank 0 depends on nothing, so if it is dirty it is re-applied alone (f = 1).
// Two attempts interact only through equal or adjacent sites, so the committed prefix is exactly
// the sequential result.  Returns the number of accepted deposits of this lane.
// ---------------------------------------------------------------------------------------------
template <int LGS, bool WRAP>
__device__ __forceinline__ uint32_t warp_run_attempts(uint32_t *sm, uint32_t A, uint32_t tile_id, uint32_t u,
                                                      uint32_t rg, uint32_t k0, uint32_t k1, uint32_t offx,
                                                      uint32_t offy, uint32_t N, uint32_t lane)
{
    using G = Geom<LGS, WRAP>;
    constexpr uint32_t S = G::S, PITCH = G::PITCH;
    const uint32_t FULL = 0xFFFFFFFFu;
    const uint32_t TAG = lane_tag(lane);
    const uint32_t nbatch = (A + 31u) >> 5;
    uint32_t my_acc = 0;
    uint32_t a0 = 0;
    // D:2 step 6: attempt a takes the 16-bit slot a & 7 of Philox call a >> 3.  Lane l computes the
    // calls 32 g + l of group g (256 attempts); attempt 32 b + l of batch b = 8 g + bb then reads
    // slot l & 7 of the call held by lane 4 bb + (l >> 3) through shuffles.
    const uint32_t sub = lane >> 3, wsel = (lane >> 1) & 3u, hsh = 16u * (lane & 1u);
    auto slot = [&](const uint4 &c, uint32_t bb) -> uint32_t {
        const uint32_t src = 4u * bb + sub;
        const uint32_t x = __shfl_sync(FULL, c.x, src), y = __shfl_sync(FULL, c.y, src);
        const uint32_t z = __shfl_sync(FULL, c.z, src), w = __shfl_sync(FULL, c.w, src);
        const uint32_t word = (wsel & 2u) ? ((wsel & 1u) ? w : z) : ((wsel & 1u) ? y : x);
        return (word >> hsh) & 0xFFFFu;
    };
    uint4 cur = philox4x32_10(lane, tile_id, u, rg, k0, k1), nxt = cur;
    uint32_t vA = slot(cur, 0u), vB = 0u;
    {
        for (uint32_t batch = 0; batch < nbatch; ++batch) {
            const uint32_t bb = batch & 7u;
            if (bb == 0u && batch + 8u < nbatch)
                nxt = philox4x32_10(32u * ((batch >> 3) + 1u) + lane, tile_id, u, rg, k0, k1);
            // vA: slots of this batch; vB: slots of the next one (lanes already past the boundary)
            if (batch + 1u < nbatch) vB = (bb < 7u) ? slot(cur, bb + 1u) : slot(nxt, 0u);
            const uint32_t batch_end = min((batch + 1u) << 5, A);
            while (a0 < batch_end) {
                const uint32_t s = a0 & 31u;
                const uint32_t rank = (lane - s) & 31u;
                const bool valid = a0 + rank < A;
                const uint32_t v = (lane >= s) ? vA : vB;
                const uint32_t X = (v & (S - 1)) + offx;
                const uint32_t Y = ((v >> LGS) & (S - 1)) + offy;
                const uint32_t px = X & 1u, py = Y & 1u, k = px | (py << 1);
                const uint32_t bx = X >> 1, by = Y >> 1;
                const uint32_t wC = by * PITCH + bx;
                uint32_t wH, wV;
                if (WRAP) {
                    wH = by * PITCH + ((bx - 1u + 2u * px) & G::NBM);
                    wV = ((by - 1u + 2u * py) & G::NBM) * PITCH + bx;
                } else {
                    wH = wC - 1u + 2u * px;
                    wV = py ? wC + PITCH : wC - PITCH;
                }
                // R
                const uint32_t C = sm[wC], H = sm[wH], V = sm[wV];
                // D: P = [C(k^1), C(k^2), H(k^1), C(k)], Q = [.., .., .., V(k^2)] -> 4 neighbours
                const uint32_t kk = k * 0x1111u;
                const uint32_t P = __byte_perm(C, H, kk ^ 0x0521u);
                const uint32_t Q = __byte_perm(P, V, (k << 12) ^ 0x6210u);
                const uint32_t t = ((P >> 24) - N) & 0x3Fu;
                const uint32_t vv = (Q & HMASK) ^ (t * 0x01010101u);
                const uint32_t z = (vv - 0x01010101u) & ~vv & 0x80808080u;   // a zero byte <=> nb == h - N
                const bool acc = valid && (z == 0u);
                const uint32_t W = (((C & HMASK) + (1u << (8u * k))) & HMASK) | TAG;
                __syncwarp();
                // W
                if (acc) sm[wC] = W;
                __syncwarp();
                // V
                const uint32_t C2 = sm[wC], H2 = sm[wH], V2 = sm[wV];
                const uint32_t selD = ((k ^ 1u) | ((k ^ 6u) << 4)) * 0x0101u;
                const uint32_t dHV = __byte_perm(H2 ^ H, V2 ^ V, selD) & HMASK;
                const bool own_ok = acc ? (C2 == W) : (((C2 ^ C) & HMASK) == 0u);
                const bool dirty = valid && (!own_ok || dHV != 0u);
                // C
                uint32_t f = __reduce_min_sync(FULL, dirty ? rank : 32u);
                if (f < 32u) {
                    // slow path: some lane is dirty
                    if (f == 0u) f = 1u;
                    const bool committed = rank < f;
                    if (acc && !committed && C2 == W) sm[wC] = C;      // undo a surviving store
                    __syncwarp();
                    if (acc && rank == 0u) sm[wC] = W;                 // rank 0 always stands
                    __syncwarp();
                    my_acc += (acc && committed) ? 1u : 0u;
                } else {
                    f = min(32u, A - a0);
                    my_acc += acc ? 1u : 0u;
                }
                a0 += f;
            }
            vA = vB;
            if (bb == 7u) cur = nxt;
        }
    }
    return my_acc;
}

__device__ __forceinline__ int32_t sext6(uint32_t d)
{
    return ((int32_t)(d << 26)) >> 26;
}

template <int LGS, bool WRAP>
__device__ __forceinline__ uint32_t sm_height(const uint32_t *sm, uint32_t X, uint32_t Y)
{
    using G = Geom<LGS, WRAP>;
    const uint8_t *b = reinterpret_cast<const uint8_t *>(sm);
    return b[((Y >> 1) * G::PITCH + (X >> 1)) * 4u + ((Y & 1u) << 1) + (X & 1u)] & 0x3Fu;
}

// ---------------------------------------------------------------------------------------------
// warp_dt: one colour pass of one sub-sweep, one warp per active tile (D:2 steps 4-6, D:4).
// ---------------------------------------------------------------------------------------------
template <int LGS>
__global__ void __launch_bounds__(WARP_DT_WARPS * 32) warp_dt_kernel(Params p, uint32_t u, uint32_t colour)
{
    using G = Geom<LGS, false>;
    constexpr uint32_t S = G::S, PITCH = G::PITCH;
    constexpr uint32_t NCH = (S + 8) / 4;            // int4 chunks per window row
    constexpr uint32_t NROW = S + 2;                 // window rows actually needed
    extern __shared__ __align__(16) uint32_t smem[];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    uint32_t *sm = smem + warp * G::WORDS;

    const uint32_t L = p.L, Lm = L - 1;
    const uint32_t T = L >> LGS, half = T >> 1, ntile = half * half;
    const uint32_t idx = blockIdx.x * WARP_DT_WARPS + warp;
    if (idx >= p.R * ntile) return;
    const uint32_t rl = idx / ntile, n = idx - rl * ntile;
    const uint32_t ti = n % half, tj = n / half;
    const uint32_t I = 2 * ti + (colour & 1u), J = 2 * tj + (colour >> 1);
    const uint32_t rg = p.first_real + rl;
    uint32_t ox, oy;
    draw_origin(p, u, rg, ox, oy);
    const uint32_t x0 = (ox + I * S) & Lm, y0 = (oy + J * S) & Lm;
    const uint32_t offx = ((x0 - 1u) & 3u) + 1u, offy = ((y0 - 1u) & 1u) + 1u;
    const uint32_t xa = (x0 - offx) & Lm;            // multiple of 4
    int32_t *h = p.h + (size_t)rl * L * L;

    // ---- stage: rows y0-1 .. y0+S, columns xa .. xa+S+7, low 6 bits of each height ----------
    {
        uint16_t *sm16 = reinterpret_cast<uint16_t *>(sm);
#pragma unroll 12
        for (uint32_t it = lane; it < NROW * NCH; it += 32u) {
            const uint32_t yr = it / NCH, c = it - yr * NCH;
            const uint32_t Y = offy - 1u + yr;
            const uint32_t gx = (xa + 4u * c) & Lm, gy = (y0 - 1u + yr) & Lm;
            const int4 q = *reinterpret_cast<const int4 *>(h + (size_t)gy * L + gx);
            const uint32_t lo = ((uint32_t)q.x & 0x3Fu) | (((uint32_t)q.y & 0x3Fu) << 8);
            const uint32_t hi = ((uint32_t)q.z & 0x3Fu) | (((uint32_t)q.w & 0x3Fu) << 8);
            const uint32_t w16 = (((Y >> 1) * PITCH + 2u * c) << 1) + (Y & 1u);   // uint16 index
            sm16[w16] = (uint16_t)lo;
            sm16[w16 + 2u] = (uint16_t)hi;
        }
    }
    __syncwarp();

    const uint32_t A = (S * S) / p.K;
    const uint32_t my_acc = warp_run_attempts<LGS, false>(sm, A, J * T + I, u, rg, p.k0, p.k1, offx, offy, p.N, lane);
    __syncwarp();

    // ---- write back: int32 heights rebuilt column by column from the frozen halo row ----------
    // h(x, y) = h(x, y-1) + sext6(b(x, y) - b(x, y-1)): adjacent heights differ by <= N <= 31.
    // All column groups of a lane advance together so that their halo loads and chains overlap.
    {
        constexpr uint32_t NG = (S + 31u) / 32u;
        int32_t hv[NG];
        uint32_t bprev[NG];
#pragma unroll
        for (uint32_t g = 0; g < NG; ++g) {
            const uint32_t cx = lane + 32u * g;
            hv[g] = 0; bprev[g] = 0;
            if (cx < S) {
                hv[g] = h[(size_t)((y0 - 1u) & Lm) * L + ((x0 + cx) & Lm)];
                bprev[g] = sm_height<LGS, false>(sm, offx + cx, offy - 1u);
            }
        }
#pragma unroll 4
        for (uint32_t dy = 0; dy < S; ++dy) {
            int32_t *grow = h + (size_t)((y0 + dy) & Lm) * L;
#pragma unroll
            for (uint32_t g = 0; g < NG; ++g) {
                const uint32_t cx = lane + 32u * g;
                if (cx < S) {
                    const uint32_t b = sm_height<LGS, false>(sm, offx + cx, offy + dy);
                    hv[g] += sext6(b - bprev[g]);
                    bprev[g] = b;
                    grow[(x0 + cx) & Lm] = hv[g];
                }
            }
        }
    }
    const uint32_t tot = __reduce_add_sync(0xFFFFFFFFu, my_acc);
    if (lane == 0 && tot) atomicAdd(p.accepted + rl, (unsigned long long)tot);
}

// ---------------------------------------------------------------------------------------------
// warp_rs: RS mode (2S > L): the schedule is serial random-sequential deposition on the whole
// lattice (D:2 step 3).  One warp per realization; the lattice is staged once, all `mcs` sweeps
// run on chip, and the int32 heights are rebuilt at the end from differences plus the exact
// identity  sum h(end) = sum h(start) + accepted.
// ---------------------------------------------------------------------------------------------
template <int LGL>
__global__ void __launch_bounds__(WARP_RS_WARPS * 32) warp_rs_kernel(Params p, uint32_t t0, uint32_t mcs)
{
    using G = Geom<LGL, true>;
    constexpr uint32_t L = G::S, PITCH = G::PITCH;
    extern __shared__ __align__(16) uint32_t smem[];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    uint32_t *sm = smem + warp * G::WORDS;
    const uint32_t rl = blockIdx.x * WARP_RS_WARPS + warp;
    if (rl >= p.R) return;
    const uint32_t rg = p.first_real + rl;
    int32_t *h = p.h + (size_t)rl * L * L;
    const uint32_t FULL = 0xFFFFFFFFu;

    // ---- stage the whole lattice; S1 = sum of the int32 heights (exact, int64) ----------------
    long long s1 = 0;
    {
        uint16_t *sm16 = reinterpret_cast<uint16_t *>(sm);
        constexpr uint32_t NCH = L / 4;
        for (uint32_t it = lane; it < L * NCH; it += 32u) {
            const uint32_t Y = it / NCH, c = it - Y * NCH;
            const int4 q = *reinterpret_cast<const int4 *>(h + (size_t)Y * L + 4u * c);
            s1 += (long long)q.x + q.y + q.z + q.w;
            const uint32_t lo = ((uint32_t)q.x & 0x3Fu) | (((uint32_t)q.y & 0x3Fu) << 8);
            const uint32_t hi = ((uint32_t)q.z & 0x3Fu) | (((uint32_t)q.w & 0x3Fu) << 8);
            const uint32_t w16 = (((Y >> 1) * PITCH + 2u * c) << 1) + (Y & 1u);
            sm16[w16] = (uint16_t)lo;
            sm16[w16 + 2u] = (uint16_t)hi;
        }
    }
    __syncwarp();

    unsigned long long my_acc = 0;
    for (uint32_t m = 0; m < mcs; ++m)
        my_acc += warp_run_attempts<LGL, true>(sm, L * L, 0u, t0 + m, rg, p.k0, p.k1, 0u, 0u, p.N, lane);
    __syncwarp();

    unsigned long long tot = my_acc;
    for (int o = 16; o; o >>= 1) {
        tot += __shfl_xor_sync(FULL, tot, o);
        s1 += __shfl_xor_sync(FULL, s1, o);
    }
    if (tot == 0ull) return;                       // nothing deposited: global heights are current

    // ---- rebuild: rel(x, y) = h(x, y) - h(0, 0) by difference chains --------------------------
    // row 0 by a warp scan along x, then every column downwards.
    constexpr uint32_t NG = (L + 31) / 32;          // column groups per lane
    int32_t rel0[NG];
    int32_t carry = 0;
#pragma unroll
    for (uint32_t g = 0; g < NG; ++g) {
        const uint32_t X = g * 32u + lane;
        int32_t d = 0;
        if (X < L && X > 0) d = sext6(sm_height<LGL, true>(sm, X, 0) - sm_height<LGL, true>(sm, X - 1u, 0));
        for (int o = 1; o < 32; o <<= 1) {
            const int32_t n = __shfl_up_sync(FULL, d, o);
            if ((int)lane >= o) d += n;
        }
        rel0[g] = d + carry;
        carry = __shfl_sync(FULL, rel0[g], 31);
    }
    long long srel = 0;
#pragma unroll
    for (uint32_t g = 0; g < NG; ++g) {
        const uint32_t X = g * 32u + lane;
        if (X < L) {
            int32_t rv = rel0[g];
            uint32_t bprev = sm_height<LGL, true>(sm, X, 0);
            srel += rv;
            for (uint32_t Y = 1; Y < L; ++Y) {
                const uint32_t b = sm_height<LGL, true>(sm, X, Y);
                rv += sext6(b - bprev);
                bprev = b;
                srel += rv;
            }
        }
    }
    for (int o = 16; o; o >>= 1) srel += __shfl_xor_sync(FULL, srel, o);
    // L^2 * h00 + srel = s1 + accepted
    const long long num = s1 + (long long)tot - srel;
    const long long h00 = num >> (2 * LGL);
    if ((h00 << (2 * LGL)) != num) { if (lane == 0) atomicOr(p.err, ERR_RECONSTRUCT); return; }
#pragma unroll
    for (uint32_t g = 0; g < NG; ++g) {
        const uint32_t X = g * 32u + lane;
        if (X < L) {
            int32_t hv = (int32_t)h00 + rel0[g];
            uint32_t bprev = sm_height<LGL, true>(sm, X, 0);
            h[X] = hv;
            for (uint32_t Y = 1; Y < L; ++Y) {
                const uint32_t b = sm_height<LGL, true>(sm, X, Y);
                hv += sext6(b - bprev);
                bprev = b;
                h[(size_t)Y * L + X] = hv;
            }
        }
    }
    if (lane == 0) atomicAdd(p.accepted + rl, tot);
}

// =============================================================================================
// Host-side launchers
// =============================================================================================
size_t warp_dt_smem(uint32_t lgS)
{
    const uint32_t S = 1u << lgS;
    return (size_t)WARP_DT_WARPS * ((S + 8) / 2) * ((S + 4) / 2) * 4;
}
size_t warp_rs_smem(uint32_t lgL)
{
    const uint32_t L = 1u << lgL;
    return (size_t)WARP_RS_WARPS * (L / 2) * (L / 2) * 4;
}

template <int LGS>
static cudaError_t launch_warp_dt_t(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st,
                                    bool configure)
{
    const size_t sm = warp_dt_smem(LGS);
    if (configure) return cudaFuncSetAttribute(warp_dt_kernel<LGS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    warp_dt_kernel<LGS><<<blocks, WARP_DT_WARPS * 32, sm, st>>>(p, u, colour);
    return cudaGetLastError();
}

static cudaError_t dispatch_warp_dt(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st,
                                    bool configure)
{
    switch (p.lgS) {
        case 3: return launch_warp_dt_t<3>(p, u, colour, blocks, st, configure);
        case 4: return launch_warp_dt_t<4>(p, u, colour, blocks, st, configure);
        case 5: return launch_warp_dt_t<5>(p, u, colour, blocks, st, configure);
        case 6: return launch_warp_dt_t<6>(p, u, colour, blocks, st, configure);
        case 7: return launch_warp_dt_t<7>(p, u, colour, blocks, st, configure);
        default: return cudaErrorInvalidValue;
    }
}

template <int LGL>
static cudaError_t launch_warp_rs_t(const Params &p, uint32_t t0, uint32_t mcs, uint32_t blocks, cudaStream_t st,
                                    bool configure)
{
    const size_t sm = warp_rs_smem(LGL);
    if (configure) return cudaFuncSetAttribute(warp_rs_kernel<LGL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    warp_rs_kernel<LGL><<<blocks, WARP_RS_WARPS * 32, sm, st>>>(p, t0, mcs);
    return cudaGetLastError();
}

static cudaError_t dispatch_warp_rs(const Params &p, uint32_t t0, uint32_t mcs, uint32_t blocks, cudaStream_t st,
                                    bool configure)
{
    switch (p.lgL) {
        case 2: return launch_warp_rs_t<2>(p, t0, mcs, blocks, st, configure);
        case 3: return launch_warp_rs_t<3>(p, t0, mcs, blocks, st, configure);
        case 4: return launch_warp_rs_t<4>(p, t0, mcs, blocks, st, configure);
        case 5: return launch_warp_rs_t<5>(p, t0, mcs, blocks, st, configure);
        case 6: return launch_warp_rs_t<6>(p, t0, mcs, blocks, st, configure);
        case 7: return launch_warp_rs_t<7>(p, t0, mcs, blocks, st, configure);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t configure_engine(const Params &p, uint32_t engine, bool mode_dt)
{
    if (engine == ENGINE_THREAD && mode_dt) return thread_dt_configure(p);
    if (engine == ENGINE_RESIDENT && mode_dt) return resident_configure(p);
    if (engine == ENGINE_FINE && mode_dt) return fine_configure(p);
    if (engine == ENGINE_MULTI && !mode_dt) return multi_configure(p);
    if (engine == ENGINE_LEVEL && !mode_dt) return level_configure(p);
    if (engine == ENGINE_WARP && mode_dt) return dispatch_warp_dt(p, 0, 0, 0, nullptr, true);
    if (engine == ENGINE_ONCHIP && !mode_dt) return dispatch_warp_rs(p, 0, 0, 0, nullptr, true);
    uint32_t pww, nrows;
    size_t gsmem;
    if (engine == ENGINE_SIMPLE && mode_dt && general_window_shape(p, &pww, &nrows, &gsmem))
        return cudaFuncSetAttribute(general_window_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gsmem);
    return cudaSuccess;
}

uint32_t engine_blocks(const Params &p, uint32_t engine, bool mode_dt)
{
    const uint32_t T = p.general ? p.T : p.L >> p.lgS, half = T >> 1;
    const uint64_t tiles = mode_dt ? (uint64_t)p.R * half * half : p.R;
    if (engine == ENGINE_THREAD) return thread_dt_blocks(p);
    if (engine == ENGINE_RESIDENT) return resident_blocks(p);
    if (engine == ENGINE_FINE) return fine_blocks(p);
    if (engine == ENGINE_MULTI) return multi_blocks(p);
    if (engine == ENGINE_LEVEL) return level_blocks(p);
    if (engine == ENGINE_WARP) return (uint32_t)((tiles + WARP_DT_WARPS - 1) / WARP_DT_WARPS);
    if (engine == ENGINE_ONCHIP) return (uint32_t)((tiles + WARP_RS_WARPS - 1) / WARP_RS_WARPS);
    return (uint32_t)((tiles + (mode_dt ? 127 : 31)) / (mode_dt ? 128 : 32));
}

// One colour pass of sub-sweep u (DT mode).
cudaError_t launch_dt_pass(const Params &p, uint32_t engine, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st)
{
    if (engine == ENGINE_THREAD) return thread_dt_launch(p, u, colour, blocks, st);
    if (engine == ENGINE_WARP) return dispatch_warp_dt(p, u, colour, blocks, st, false);
    uint32_t pww, nrows;
    size_t gsmem;
    if (general_window_shape(p, &pww, &nrows, &gsmem)) {               // general L, N <= 7: tile windows in shared memory
        const uint32_t half = p.T >> 1;
        const uint64_t tiles = (uint64_t)p.R * half * half;
        general_window_kernel<<<(uint32_t)((tiles + GW_NT - 1) / GW_NT), 32, gsmem, st>>>(p, u, colour, pww, nrows);
        return cudaGetLastError();
    }
    simple_dt_kernel<<<blocks, 128, 0, st>>>(p, u, colour);
    return cudaGetLastError();
}

// `mcs` whole sweeps starting at sweep counter t0 (RS mode).
cudaError_t launch_rs_sweeps(const Params &p, uint32_t engine, uint32_t t0, uint32_t mcs, uint32_t blocks, cudaStream_t st)
{
    if (engine == ENGINE_ONCHIP) return dispatch_warp_rs(p, t0, mcs, blocks, st, false);
    if (engine == ENGINE_MULTI) return multi_launch(p, t0, mcs, st);
    if (engine == ENGINE_LEVEL) return level_launch(p, t0, mcs, st);
    simple_rs_kernel<<<blocks, 32, 0, st>>>(p, t0, mcs);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// Philox test hook (rsos_philox): the same device function on n (counter, key) pairs.
// ---------------------------------------------------------------------------------------------
__global__ void philox_kernel(const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint32_t n)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint4 o = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1]);
    out[4 * i] = o.x; out[4 * i + 1] = o.y; out[4 * i + 2] = o.z; out[4 * i + 3] = o.w;
}

cudaError_t launch_philox(const uint32_t *d_ctr, const uint32_t *d_key, uint32_t *d_out, uint32_t n, cudaStream_t st)
{
    philox_kernel<<<(n + 255) / 256, 256, 0, st>>>(d_ctr, d_key, d_out, n);
    return cudaGetLastError();
}

}  // namespace rsos
