/*
 * rsos_oracle.c -- CPU ORACLE for the RSOS deposition Monte Carlo of arxiv 1605.02620.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or helper with the CUDA path under paper_1605_02620_b200/csrc/.
 *
 * Plain, slow, literal.  Every function cites the passage it follows:
 *   P:n   = /root/reference/PAPER.md line n  (with section / equation)
 *   S8c.1 = SURVEY.md section 8(c).1, the seeded schedule DT(S,K) / RS (restated in DESIGN.md)
 *
 * What the paper fixes (and this file writes out):
 *   - RSOS rule, Eq. (6): "deposition at random sites if the local height difference
 *     satisfies |h(x,t) - h(x',t)| <= N".  Reading Q1: a deposit h(x) += 1 is
 *     accepted iff afterwards |h(x) - h(x')| <= N for the four nearest neighbours x'
 *     (periodic, reading Q2); a rejected deposit changes nothing but still counts (Q3).
 *   - flat start h = 0, time in Monte-Carlo steps; 1 MCS = L*L attempts (Q4).
 *   - squared interface width, Eq. (2), P:40-43:
 *         W2 = (1/L^2) sum h^2 - ((1/L^2) sum h)^2.
 *   - domain decomposition by double tiling with an origin moved randomly after each
 *     sweep; independent realizations.
 * What the paper leaves open (tile size, colour order, RNG, slot layout) is fixed by S8c.1.
 * Lattice sides that are not powers of two (the paper's L = 9605; irregular tilings)
 * follow the general-L schedule DTG / RSG of DESIGN.md section 2b: tiles of two sizes that divide
 * the lattice, sites drawn by an exactly uniform bounded draw (multiply-shift with rejection).
 *
 * Pins (tests/test_oracle_*.py, all CPU): Eq. (6) invariant after every attempt, monotone
 * heights, sum h == accepted, random-deposition closed form, exact Markov-chain enumeration
 * on 2x2 / 4x4 (+3x3 through the general-L draw), Philox known answers + cuRAND header,
 * DT-vs-RS statistical agreement, tile-order independence, W2 recomputed with rationals;
 * moments (Eq. 13-15): hand-worked 2x2 examples, scipy.stats, exact rationals.
 * "Parity unpinned": the schedule's free choices (S, colour order, slot layout, origin range)
 * cannot be pinned by the paper; they are pinned by oracle == GPU equality plus the
 * DT-vs-RS statistical test only.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------
 * Philox4x32 with 10 rounds (Salmon, Moraes, Dror, Shaw, SC'11), the published algorithm.
 * One round:  (hi0,lo0) = M0 * c0 ;  (hi1,lo1) = M1 * c2 ;
 *             c <- ( hi1 ^ c1 ^ k0 ,  lo1 ,  hi0 ^ c3 ^ k1 ,  lo0 )
 * and the key is bumped by the Weyl constants (W0, W1) between rounds.
 * S8c.1 step 2.
 * ------------------------------------------------------------------------------------------ */
void rsos_oracle_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------------------------------
 * One deposition attempt at site (x, y) of one L x L surface h (row-major, h[y*L + x]).
 * Eq. (6) P:61-63 with readings Q1-Q3; S8c.1 step 6, last bullet.  The four tests are the
 * literal absolute-value ones.  Works for any L >= 1 (for L = 2 left == right neighbour).
 * Returns 1 if the deposit was accepted.
 * ------------------------------------------------------------------------------------------ */
int rsos_oracle_attempt(int32_t *h, uint32_t L, int64_t N, uint32_t x, uint32_t y)
{
    uint32_t xm = (x + L - 1) % L, xp = (x + 1) % L;
    uint32_t ym = (y + L - 1) % L, yp = (y + 1) % L;
    int64_t c = (int64_t)h[(size_t)y * L + x] + 1;
    int64_t d;
    d = c - h[(size_t)y * L + xm];  if (d < 0) d = -d;  if (d > N) return 0;
    d = c - h[(size_t)y * L + xp];  if (d < 0) d = -d;  if (d > N) return 0;
    d = c - h[(size_t)ym * L + x];  if (d < 0) d = -d;  if (d > N) return 0;
    d = c - h[(size_t)yp * L + x];  if (d < 0) d = -d;  if (d > N) return 0;
    h[(size_t)y * L + x] = (int32_t)c;
    return 1;
}

/* Eq. (6) on every bond of one surface: returns the number of violated bonds (0 = valid). */
int64_t rsos_oracle_violations(const int32_t *h, uint32_t L, int64_t N)
{
    int64_t bad = 0;
    for (uint32_t y = 0; y < L; ++y)
        for (uint32_t x = 0; x < L; ++x) {
            int64_t a = h[(size_t)y * L + x];
            int64_t r = h[(size_t)y * L + (x + 1) % L];
            int64_t u = h[(size_t)((y + 1) % L) * L + x];
            int64_t d1 = a - r, d2 = a - u;
            if (d1 < 0) d1 = -d1;
            if (d2 < 0) d2 = -d2;
            bad += (d1 > N) + (d2 > N);
        }
    return bad;
}

/* ------------------------------------------------------------------------------------------
 * Context.  S8c.1 step 1: per realization int32 h[L][L] and int64 accepted; sweep counter t.
 * ------------------------------------------------------------------------------------------ */
typedef struct rsos_oracle {
    uint32_t L, R, S, K, first_real;
    int64_t  N;
    uint64_t seed, t;
    int      mode_dt;        /* 1 = DT(S,K) (DTG when L is not a power of two), 0 = RS (2S > L) */
    int      pow2;           /* L is a power of two                                          */
    uint32_t T;              /* general-L DT mode: tiles per side (even); 0 otherwise        */
    int      poisson;        /* 1 = DTP(c): Poisson(4) attempts per cell and sub-sweep (D:2c) */
    int      multisurface;   /* 1 = MS: shared-coordinate multisurface schedule (D:2d)  */
    uint32_t lgL, lgS;
    int32_t *h;              /* R * L * L                                                    */
    int64_t *accepted;       /* R                                                            */
    /* debug switches (tests only) */
    int      check_each;     /* verify Eq. (6) + monotonicity after every attempt (P1, P2)   */
    uint64_t shuffle_seed;   /* != 0: visit same-colour tiles in a shuffled order (P8)        */
    int64_t  violations;     /* accumulated by check_each                                    */
    int      threads;        /* OpenMP threads to use (0 = default)                          */
} rsos_oracle;

static int is_pow2(uint32_t v) { return v && !(v & (v - 1)); }
static uint32_t ilog2(uint32_t v) { uint32_t l = 0; while ((1u << l) < v) ++l; return l; }

static char g_err[256];
const char *rsos_oracle_last_error(void) { return g_err; }

/* ------------------------------------------------------------------------------------------
 * Create / free.  S8c.1 steps 1 and 3.  S = tile side, K = sub-sweeps per MCS.
 *   mode RS  when 2*S > L;  mode DT  otherwise; needs S, K powers of two, K | S*S, S*S/K >= 32.
 *   L not a power of two: the general-L forms RSG / DTG of the same two modes (D:2b).
 * All heights 0, accepted 0, t = 0 (flat start).
 * ------------------------------------------------------------------------------------------ */
rsos_oracle *rsos_oracle_create(uint32_t L, int64_t N, uint32_t R, uint64_t seed,
                                uint32_t S, uint32_t K, uint32_t first_real)
{
    g_err[0] = 0;
    if (L < 2 || N < 1 || R == 0) { snprintf(g_err, sizeof g_err, "bad L/N/R"); return NULL; }
    if (S == 0) S = 64;
    if (K == 0) K = 1;
    rsos_oracle *c = (rsos_oracle *)calloc(1, sizeof *c);
    if (!c) return NULL;
    c->L = L; c->N = N; c->R = R; c->seed = seed; c->first_real = first_real;
    c->pow2 = is_pow2(L);
    c->lgL = ilog2(L);
    if (2 * (uint64_t)S > L) {                      /* RS: one tile = the whole lattice */
        c->mode_dt = 0; c->S = L; c->K = 1; c->lgS = c->lgL;
    } else if (!c->pow2) {                          /* DTG: D:2b, T = 2 floor(L / 2S) tiles per side */
        if (!is_pow2(S) || S < 8 || !is_pow2(K) || ((uint64_t)S * S) % K || (uint64_t)S * S / K < 32) {
            snprintf(g_err, sizeof g_err, "bad S/K"); free(c); return NULL;
        }
        c->mode_dt = 1; c->S = S; c->K = K; c->lgS = ilog2(S); c->T = 2 * (L / (2 * S));
    } else {
        if (!is_pow2(S) || S < 8 || !is_pow2(K) || ((uint64_t)S * S) % K || (uint64_t)S * S / K < 32) {
            snprintf(g_err, sizeof g_err, "bad S/K"); free(c); return NULL;
        }
        c->mode_dt = 1; c->S = S; c->K = K; c->lgS = ilog2(S);
    }
    c->h = (int32_t *)calloc((size_t)R * L * L, sizeof(int32_t));
    c->accepted = (int64_t *)calloc(R, sizeof(int64_t));
    if (!c->h || !c->accepted) { free(c->h); free(c->accepted); free(c);
        snprintf(g_err, sizeof g_err, "out of memory"); return NULL; }
    return c;
}

void rsos_oracle_free(rsos_oracle *c) { if (c) { free(c->h); free(c->accepted); free(c); } }

void rsos_oracle_set_debug(rsos_oracle *c, int check_each, uint64_t shuffle_seed, int threads)
{ c->check_each = check_each; c->shuffle_seed = shuffle_seed; c->threads = threads; }

int64_t rsos_oracle_debug_violations(const rsos_oracle *c) { return c->violations; }
int rsos_oracle_mode_dt(const rsos_oracle *c) { return c->mode_dt; }

/* One attempt with the optional per-attempt checks P1 (Eq. 6 at the touched bonds; all other
 * bonds are unchanged) and P2 (height changes by exactly +1 on accept, 0 on reject). */
static int attempt_checked(rsos_oracle *c, int32_t *h, uint32_t x, uint32_t y)
{
    if (!c->check_each) return rsos_oracle_attempt(h, c->L, c->N, x, y);
    uint32_t L = c->L;
    int32_t before = h[(size_t)y * L + x];
    int acc = rsos_oracle_attempt(h, L, c->N, x, y);
    int64_t now = h[(size_t)y * L + x];
    int64_t bad = (now != (int64_t)before + acc);
    int64_t nb[4] = { h[(size_t)y * L + (x + L - 1) % L], h[(size_t)y * L + (x + 1) % L],
                      h[(size_t)((y + L - 1) % L) * L + x], h[(size_t)((y + 1) % L) * L + x] };
    for (int i = 0; i < 4; ++i) { int64_t d = now - nb[i]; if (d < 0) d = -d; bad += (d > c->N); }
    if (bad) {
#ifdef _OPENMP
#pragma omp atomic
#endif
        c->violations += bad;
    }
    return acc;
}

/* ------------------------------------------------------------------------------------------
 * All A attempts of one tile, in order a = 0 .. A-1.  S8c.1 step 6:
 *   slot width w = 16 if 2*lg(Se) <= 16 else 32; ns = 128/w slots per Philox call;
 *   q = a / ns (call index), j = a % ns (slot within the call): consecutive attempts consume
 *   the slots of one call in order, then the next call (DESIGN.md section 2 step 6, reading Q16);
 *   o = Philox(counter = (q, tile id, u, r), key = seed);
 *   v = 16-bit slot j of o (low half first) or o[j];  dx = v & (Se-1), dy = (v >> lg Se) & (Se-1);
 *   site x = (ox + I*S + dx) & (L-1), y = (oy + J*S + dy) & (L-1).
 * (Lattice sides that are not powers of two never come here: run_tile_general.)
 * Returns the number of accepted deposits.
 * ------------------------------------------------------------------------------------------ */
static int64_t run_tile(rsos_oracle *c, int32_t *h, uint32_t rg, uint32_t u, uint32_t tile_id,
                        uint32_t x0, uint32_t y0, uint32_t Se, uint32_t lgSe, uint64_t A)
{
    const uint32_t L = c->L;
    const uint32_t key[2] = { (uint32_t)(c->seed & 0xffffffffu), (uint32_t)(c->seed >> 32) };
    const uint32_t w = (2 * lgSe <= 16) ? 16 : 32;
    const uint32_t ns = 128 / w;
    int64_t acc = 0;
    uint64_t a = 0;
    for (uint64_t q = 0; a < A; ++q) {
        uint32_t ctr[4] = { (uint32_t)q, tile_id, u, rg }, o[4];
        rsos_oracle_philox(ctr, key, o);
        for (uint32_t j = 0; j < ns && a < A; ++j, ++a) {
            uint32_t v = (w == 16) ? (o[j >> 1] >> (16 * (j & 1))) & 0xffffu : o[j];
            uint32_t dx = v & (Se - 1), dy = (v >> lgSe) & (Se - 1);
            uint32_t x = (x0 + dx) & (L - 1);
            uint32_t y = (y0 + dy) & (L - 1);
            acc += attempt_checked(c, h, x, y);
        }
    }
    return acc;
}

/* ------------------------------------------------------------------------------------------
 * General-L schedule, for lattice sides that are not powers of two.
 *
 * Word stream of (tile id, u, r): word i = o[i & 3] of Philox(counter (i >> 2, tile id, u, r)).
 * draw(n), exactly uniform on [0, n) (Lemire's multiply-shift with rejection in its plain form):
 *     thr = 2^32 mod n;  repeat  v = next word;  m = v * n (64 bit)  until (m mod 2^32) >= thr;
 *     return m >> 32.
 * Every value of [0, n) is hit by exactly floor(2^32 / n) of the 2^32 words (pinned by a census
 * over all words, tests/test_oracle_general.py); a rejected word (probability < n / 2^32) is
 * skipped and the next word of the stream is taken.
 * ------------------------------------------------------------------------------------------ */
typedef struct { uint32_t ctr[4], key[2], o[4]; uint32_t j; } word_stream;

static void stream_init(word_stream *s, const rsos_oracle *c, uint32_t tile_id, uint32_t u, uint32_t rg)
{
    s->ctr[0] = 0; s->ctr[1] = tile_id; s->ctr[2] = u; s->ctr[3] = rg;
    s->key[0] = (uint32_t)(c->seed & 0xffffffffu); s->key[1] = (uint32_t)(c->seed >> 32);
    s->j = 4;                                   /* nothing generated yet */
}

static uint32_t stream_next(word_stream *s)
{
    if (s->j == 4) { rsos_oracle_philox(s->ctr, s->key, s->o); s->ctr[0] += 1; s->j = 0; }
    return s->o[s->j++];
}

uint32_t rsos_oracle_bounded(uint32_t v, uint32_t n, int *accepted)
{
    const uint32_t thr = (uint32_t)(0x100000000ull % n);
    const uint64_t m = (uint64_t)v * n;
    *accepted = (uint32_t)m >= thr;
    return (uint32_t)(m >> 32);
}

static uint32_t stream_draw(word_stream *s, uint32_t n)
{
    for (;;) {
        int ok;
        const uint32_t r = rsos_oracle_bounded(stream_next(s), n, &ok);
        if (ok) return r;
    }
}

/* Census of draw(n) over ALL 2^32 words (test hook): counts[v] = words mapped to v, *rejected = words
 * rejected.  Exact uniformity means counts[v] == floor(2^32 / n) for every v and *rejected == 2^32 mod n. */
void rsos_oracle_bounded_census(uint32_t n, uint64_t *counts, uint64_t *rejected)
{
    uint64_t rej = 0;
    for (uint32_t v = 0; v < n; ++v) counts[v] = 0;
#ifdef _OPENMP
#pragma omp parallel
#endif
    {
        uint64_t *loc = (uint64_t *)calloc(n, sizeof(uint64_t));
        uint64_t lrej = 0;
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int64_t w = 0; w < 0x100000000ll; ++w) {
            int ok;
            const uint32_t r = rsos_oracle_bounded((uint32_t)w, n, &ok);
            if (ok) loc[r] += 1; else lrej += 1;
        }
#ifdef _OPENMP
#pragma omp critical
#endif
        { for (uint32_t v = 0; v < n; ++v) counts[v] += loc[v]; rej += lrej; }
        free(loc);
    }
    *rejected = rej;
}

/* Boundary of tile column / row i of T on a lattice of side L: floor(i * L / T)  (D:2b). */
static uint32_t tile_edge(uint32_t i, uint32_t L, uint32_t T) { return (uint32_t)(((uint64_t)i * L) / T); }

/* All A attempts of one general tile of w x hgt sites whose first site is (x0, y0), in order:
 *   s = draw(w * hgt);  dx = s mod w, dy = s div w;  site ((x0 + dx) mod L, (y0 + dy) mod L).   D:2b. */
static int64_t run_tile_general(rsos_oracle *c, int32_t *h, uint32_t rg, uint32_t u, uint32_t tile_id,
                                uint32_t x0, uint32_t y0, uint32_t w, uint32_t hgt, uint64_t A)
{
    const uint32_t L = c->L;
    word_stream st;
    stream_init(&st, c, tile_id, u, rg);
    int64_t acc = 0;
    for (uint64_t a = 0; a < A; ++a) {
        const uint32_t s = stream_draw(&st, w * hgt);
        const uint32_t dx = s % w, dy = s / w;
        acc += attempt_checked(c, h, (x0 + dx) % L, (y0 + dy) % L);
    }
    return acc;
}

/* One MCS of the general-L schedule (D:2b).  RSG: one tile = the lattice, origin (0, 0), L*L attempts.
 * DTG: T = 2 floor(L / 2S) tiles per side with edges floor(i L / T); for k < K: u = t K + k; origin
 * (ox, oy) = (draw(L), draw(L)) from the stream of tile id 0xFFFFFFFF; colours 0..3 as in DT; tile
 * (I, J) of n = w * hgt sites makes floor((k+1) n / K) - floor(k n / K) attempts in sub-sweep k (n per MCS). */
static void one_mcs_general(rsos_oracle *c, uint32_t rl, uint64_t t, int par_tiles)
{
    const uint32_t L = c->L, K = c->K, T = c->T;
    int32_t *h = c->h + (size_t)rl * L * L;
    const uint32_t rg = c->first_real + rl;
    if (!c->mode_dt) {
        c->accepted[rl] += run_tile_general(c, h, rg, (uint32_t)t, 0, 0, 0, L, L, (uint64_t)L * L);
        return;
    }
    const uint32_t half = T / 2, ntile = half * half;
    for (uint32_t k = 0; k < K; ++k) {
        const uint32_t u = (uint32_t)(t * K + k);
        word_stream os;
        stream_init(&os, c, 0xFFFFFFFFu, u, rg);
        const uint32_t ox = stream_draw(&os, L);
        const uint32_t oy = stream_draw(&os, L);
        for (uint32_t p = 0; p < 4; ++p) {
            int64_t acc = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 4) reduction(+:acc) if (par_tiles)
#endif
            for (uint32_t n = 0; n < ntile; ++n) {
                const uint32_t I = 2 * (n % half) + (p & 1), J = 2 * (n / half) + (p >> 1);
                const uint32_t bx = tile_edge(I, L, T), by = tile_edge(J, L, T);
                const uint32_t w = tile_edge(I + 1, L, T) - bx, hgt = tile_edge(J + 1, L, T) - by;
                const uint64_t sites = (uint64_t)w * hgt;
                const uint64_t A = ((uint64_t)(k + 1) * sites) / K - ((uint64_t)k * sites) / K;
                acc += run_tile_general(c, h, rg, u, J * T + I, (ox + bx) % L, (oy + by) % L, w, hgt, A);
            }
            c->accepted[rl] += acc;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Poisson variant DTP(c) of the DT schedule ("16 passes per MCS,
 * new origin per pass, Poisson(4) attempts per cell per pass ... matches serial"): K = c*c/4 sub-sweeps
 * per MCS, each with its own origin, and in every sub-sweep a cell makes n attempts with n drawn from
 * the Poisson distribution of mean 4 instead of exactly c*c/K = 4.  The count comes from the first
 * word w of Philox(counter (0xFFFFFFFF, tile id, u, r)) by inversion with the 32-bit table
 *     POISSON4[k] = floor(2^32 * P(X <= k)),  X ~ Poisson(4),  k = 0 .. 22:   n = #{k : w >= POISSON4[k]}
 * (so P(n <= k) = POISSON4[k] / 2^32; the table is pinned against a 60-digit evaluation in
 * tests/test_oracle_poisson.py).  The n attempts then take the slots 0 .. n-1 of the cell exactly as in DT
 * (slot a mod 8 of call a div 8).  Thinning: every site of the cell gets Poisson(4 / c^2) attempts per
 * sub-sweep, independently of the others -- Poisson(1) per MCS, which is what serial random-sequential
 * deposition gives in the large-lattice limit; the fixed count of DT gives Binomial(c^2, 1/c^2).
 * ------------------------------------------------------------------------------------------ */
static const uint32_t POISSON4[23] = {
    78665070u, 393325350u, 1022645910u, 1861739990u, 2700834071u, 3372109335u, 3819626178u, 4075350088u,
    4203212043u, 4260039579u, 4282770593u, 4291036416u, 4293791691u, 4294639467u, 4294881689u, 4294946282u,
    4294962430u, 4294966230u, 4294967074u, 4294967252u, 4294967287u, 4294967294u, 4294967295u };

uint32_t rsos_oracle_poisson4(uint32_t w)
{
    uint32_t n = 0;
    for (int k = 0; k < 23; ++k) n += (w >= POISSON4[k]);
    return n;
}

int rsos_oracle_set_poisson(rsos_oracle *c, int on)
{
    if (on && (!c->mode_dt || !c->pow2)) { snprintf(g_err, sizeof g_err, "DTP needs DT mode on a power-of-two lattice"); return -1; }
    c->poisson = on ? 1 : 0;
    if (on) c->K = c->S * c->S / 4;                 /* mean 4 attempts per cell and sub-sweep */
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Shared-coordinate multisurface schedule MS.  P:75: "Each single instruction
 * multiple thread (SIMT) unit of the GPU updates 128 realizations, in which the sequence of randomly
 * selected coordinates for update is the same.  This correlation was broken by updating only half of
 * the selected lattice sites in each attempt."  Reading Q5 (the paper does not say which half, nor how
 * time is counted):
 *   - realizations are grouped by their GLOBAL index: group g = r div 128, member b = r mod 128;
 *   - in sweep t the group draws 2 L^2 coordinates, selection a = 0 .. 2 L^2 - 1 in order, from the
 *     coordinate stream Philox(counter (q, 0xFFFFFFFD, t, g)) with the slot layout of RS (D:2 step 6);
 *   - member b attempts the deposit at selection a iff bit (b mod 32) of word (b div 32) of
 *     Philox(counter (a, 0xFFFFFFFC, t, g)) is 1: an independent fair bit per member and selection, so
 *     each surface makes L^2 attempts per MCS on average;
 *   - whole lattice, no decomposition (2S > L), L a power of two.
 * A realization is still a pure function of (seed, r, t): this function follows one realization alone.
 * ------------------------------------------------------------------------------------------ */
static void one_mcs_multisurface(rsos_oracle *c, uint32_t rl, uint64_t t)
{
    const uint32_t L = c->L, lgL = c->lgL;
    int32_t *h = c->h + (size_t)rl * L * L;
    const uint32_t rg = c->first_real + rl, g = rg >> 7, b = rg & 127u;
    const uint32_t key[2] = { (uint32_t)(c->seed & 0xffffffffu), (uint32_t)(c->seed >> 32) };
    const uint32_t w = (2 * lgL <= 16) ? 16 : 32, ns = 128 / w;
    const uint64_t A = 2ull * L * L;
    uint32_t co[4] = { 0, 0, 0, 0 };
    int64_t acc = 0;
    for (uint64_t a = 0; a < A; ++a) {
        const uint32_t j = (uint32_t)(a % ns);
        if (j == 0) { uint32_t cc[4] = { (uint32_t)(a / ns), 0xFFFFFFFDu, (uint32_t)t, g }; rsos_oracle_philox(cc, key, co); }
        const uint32_t v = (w == 16) ? (co[j >> 1] >> (16 * (j & 1))) & 0xffffu : co[j];
        const uint32_t x = v & (L - 1), y = (v >> lgL) & (L - 1);
        uint32_t mc[4] = { (uint32_t)a, 0xFFFFFFFCu, (uint32_t)t, g }, mo[4];
        rsos_oracle_philox(mc, key, mo);
        if ((mo[b >> 5] >> (b & 31u)) & 1u) acc += attempt_checked(c, h, x, y);
    }
    c->accepted[rl] += acc;
}

int rsos_oracle_set_multisurface(rsos_oracle *c, int on)
{
    if (on && (c->mode_dt || !c->pow2 || 2ull * c->L * c->L >= (1ull << 32))) {
        snprintf(g_err, sizeof g_err, "MS needs RS mode on a power-of-two lattice"); return -1; }
    c->multisurface = on ? 1 : 0;
    return 0;
}

static uint64_t splitmix64(uint64_t *s)
{ uint64_t z = (*s += 0x9E3779B97F4A7C15ull); z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull; return z ^ (z >> 31); }

/* ------------------------------------------------------------------------------------------
 * One MCS of realization rl (local index) at sweep counter t.  S8c.1 steps 3-6.
 * DT: for k < K: u = t*K + k; origin (ox, oy) = Philox(counter (0, 0xFFFFFFFF, u, r)) & (L-1);
 *     for colour p = 0..3: every tile (I,J) with (I&1) + 2*(J&1) == p, id = J*T + I.
 * Tiles of one colour are >= S sites apart and an attempt reads only distance <= 1, so their
 * order is irrelevant (checked by the shuffle pin P8) and they may run on different threads.
 * ------------------------------------------------------------------------------------------ */
static void one_mcs(rsos_oracle *c, uint32_t rl, uint64_t t, int par_tiles)
{
    const uint32_t L = c->L, S = c->S, K = c->K;
    int32_t *h = c->h + (size_t)rl * L * L;
    const uint32_t rg = c->first_real + rl;
    if (!c->pow2) { one_mcs_general(c, rl, t, par_tiles); return; }
    if (c->multisurface) { one_mcs_multisurface(c, rl, t); return; }
    if (!c->mode_dt) {
        c->accepted[rl] += run_tile(c, h, rg, (uint32_t)t, 0, 0, 0, L, c->lgL, (uint64_t)L * L);
        return;
    }
    const uint32_t T = L / S, half = T / 2, ntile = half * half;
    const uint64_t A_fixed = (uint64_t)S * S / K;
    const uint32_t key[2] = { (uint32_t)(c->seed & 0xffffffffu), (uint32_t)(c->seed >> 32) };
    uint32_t *order = (uint32_t *)malloc(sizeof(uint32_t) * ntile);
    for (uint32_t k = 0; k < K; ++k) {
        const uint32_t u = (uint32_t)(t * K + k);
        uint32_t octr[4] = { 0, 0xFFFFFFFFu, u, rg }, o[4];
        rsos_oracle_philox(octr, key, o);
        const uint32_t ox = o[0] & (L - 1), oy = o[1] & (L - 1);
        for (uint32_t p = 0; p < 4; ++p) {
            for (uint32_t n = 0; n < ntile; ++n) order[n] = n;
            if (c->shuffle_seed) {
                uint64_t s = c->shuffle_seed ^ ((uint64_t)u << 8) ^ p ^ ((uint64_t)rg << 40);
                for (uint32_t n = ntile; n > 1; --n) {
                    uint32_t m = (uint32_t)(splitmix64(&s) % n);
                    uint32_t tmp = order[n - 1]; order[n - 1] = order[m]; order[m] = tmp;
                }
            }
            int64_t acc = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 4) reduction(+:acc) if (par_tiles)
#endif
            for (uint32_t n = 0; n < ntile; ++n) {
                uint32_t i = order[n] % half, j = order[n] / half;
                uint32_t I = 2 * i + (p & 1), J = 2 * j + (p >> 1);
                uint32_t x0 = (ox + I * S) & (L - 1), y0 = (oy + J * S) & (L - 1);
                uint64_t A = A_fixed;
                if (c->poisson) {                   /* D:2c: the cell's attempt count of this sub-sweep */
                    uint32_t cctr[4] = { 0xFFFFFFFFu, J * T + I, u, rg }, co[4];
                    rsos_oracle_philox(cctr, key, co);
                    A = rsos_oracle_poisson4(co[0]);
                }
                acc += run_tile(c, h, rg, u, J * T + I, x0, y0, S, c->lgS, A);
            }
            c->accepted[rl] += acc;
        }
    }
    free(order);
}

/* Advance all realizations by `mcs` Monte-Carlo steps (1 MCS = L*L attempts each, Q4). */
int rsos_oracle_advance(rsos_oracle *c, uint64_t mcs)
{
    if ((c->t + mcs) * c->K >= (1ull << 32)) { snprintf(g_err, sizeof g_err, "t*K overflows 2^32"); return -1; }
    int nthr = 1;
#ifdef _OPENMP
    nthr = c->threads > 0 ? c->threads : omp_get_max_threads();
    omp_set_num_threads(nthr);
#endif
    if (c->R >= (uint32_t)nthr || !c->mode_dt || nthr == 1) {
        /* realizations are independent: one thread follows one realization in time */
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1)
#endif
        for (uint32_t r = 0; r < c->R; ++r)
            for (uint64_t m = 0; m < mcs; ++m) one_mcs(c, r, c->t + m, 0);
    } else {
        for (uint32_t r = 0; r < c->R; ++r)
            for (uint64_t m = 0; m < mcs; ++m) one_mcs(c, r, c->t + m, 1);
    }
    c->t += mcs;
    return 0;
}

int rsos_oracle_threads(const rsos_oracle *c)
{
#ifdef _OPENMP
    return c->threads > 0 ? c->threads : omp_get_max_threads();
#else
    (void)c; return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * Width.  Eq. (2), S8c.1 step 7.  S1 = sum h (int64), S2 = sum h^2 (uint64);
 * W2 = (L^2 * S2 - S1^2) / L^4 evaluated from one exact 128-bit numerator.
 * ------------------------------------------------------------------------------------------ */
int rsos_oracle_sums(const rsos_oracle *c, int64_t *S1, uint64_t *S2, int64_t *accepted)
{
    const size_t n = (size_t)c->L * c->L;
    for (uint32_t r = 0; r < c->R; ++r) {
        const int32_t *h = c->h + r * n;
        int64_t s1 = 0; uint64_t s2 = 0;
        for (size_t i = 0; i < n; ++i) { int64_t v = h[i]; s1 += v; s2 += (uint64_t)(v * v); }
        if (S1) S1[r] = s1;
        if (S2) S2[r] = s2;
        if (accepted) accepted[r] = c->accepted[r];
    }
    return 0;
}

int rsos_oracle_width(const rsos_oracle *c, double *W2, double *hmean)
{
    const double n = (double)c->L * (double)c->L;
    const unsigned __int128 n_int = (unsigned __int128)c->L * c->L;
    for (uint32_t r = 0; r < c->R; ++r) {
        int64_t s1; uint64_t s2;
        const int32_t *h = c->h + (size_t)r * c->L * c->L;
        s1 = 0; s2 = 0;
        for (size_t i = 0; i < (size_t)c->L * c->L; ++i) { int64_t v = h[i]; s1 += v; s2 += (uint64_t)(v * v); }
        unsigned __int128 a1 = (unsigned __int128)(s1 < 0 ? -s1 : s1);
        unsigned __int128 num = n_int * s2 - a1 * a1;      /* >= 0 by Cauchy-Schwarz */
        if (W2) W2[r] = (double)num / (n * n);
        if (hmean) hmean[r] = (double)s1 / n;
    }
    return 0;
}

/* State access (snapshot / restart; realization is a pure function of (seed, r, L, N, S, K)). */
int rsos_oracle_get_heights(const rsos_oracle *c, uint32_t r0, uint32_t nr, int32_t *out)
{
    if ((uint64_t)r0 + nr > c->R) return -1;
    memcpy(out, c->h + (size_t)r0 * c->L * c->L, (size_t)nr * c->L * c->L * sizeof(int32_t));
    return 0;
}

int rsos_oracle_set_state(rsos_oracle *c, uint32_t r0, uint32_t nr, const int32_t *in,
                          uint64_t t, const int64_t *accepted)
{
    if ((uint64_t)r0 + nr > c->R) return -1;
    memcpy(c->h + (size_t)r0 * c->L * c->L, in, (size_t)nr * c->L * c->L * sizeof(int32_t));
    c->t = t;
    if (accepted) memcpy(c->accepted + r0, accepted, nr * sizeof(int64_t));
    return 0;
}

uint64_t rsos_oracle_time(const rsos_oracle *c) { return c->t; }
int32_t *rsos_oracle_heights_ptr(rsos_oracle *c) { return c->h; }

/* ------------------------------------------------------------------------------------------
 * Moments of the height distribution of ONE surface.  Eq. (13) P:180-184 with the observable
 * phi = h(x) and P_L the empirical distribution of the L*L heights of realization r:
 *     hbar   = (1/L^2) sum_x h(x)
 *     Phi^n  = (1/L^2) sum_x (h(x) - hbar)^n ,   n = 2, 3, 4
 * written out as the definition: two passes in floating point (long double accumulators), no
 * algebraic expansion into raw power sums.  out[0..2] = Phi^2, Phi^3, Phi^4; *hbar_out = hbar.
 * The skewness Eq. (14) and kurtosis Eq. (15) of an ensemble are
 *     S = <Phi^3> / <Phi^2>^(3/2),   Q = <Phi^4> / <Phi^2>^2 - 3
 * with <.> the average over surfaces (and times) -- formed by the caller from these values.
 * Pins (tests/test_oracle_moments.py): hand-worked 2x2 examples, scipy.stats moment/skew/kurtosis.
 * ------------------------------------------------------------------------------------------ */
int rsos_oracle_height_moments(const rsos_oracle *c, uint32_t r, double out[3], double *hbar_out)
{
    if (r >= c->R) return -1;
    const size_t n = (size_t)c->L * c->L;
    const int32_t *h = c->h + (size_t)r * n;
    long double s = 0.0L;
    for (size_t i = 0; i < n; ++i) s += (long double)h[i];
    const long double hbar = s / (long double)n;
    long double p2 = 0.0L, p3 = 0.0L, p4 = 0.0L;
    for (size_t i = 0; i < n; ++i) {
        const long double d = (long double)h[i] - hbar;
        p2 += d * d;
        p3 += d * d * d;
        p4 += d * d * d * d;
    }
    out[0] = (double)(p2 / (long double)n);
    out[1] = (double)(p3 / (long double)n);
    out[2] = (double)(p4 / (long double)n);
    if (hbar_out) *hbar_out = (double)hbar;
    return 0;
}

/* Exact integer power sums about an integer base b:  M_k = sum_x (h(x) - b)^k, k = 1..4, as signed
 * 128-bit integers, each written as two uint64 words (lo, hi).  This is the quantity the C ABI's
 * rsos_moments returns (with b = floor(S1 / L^2)); the definition written out, one site at a time. */
int rsos_oracle_power_sums(const rsos_oracle *c, uint32_t r, int64_t base, uint64_t out[8])
{
    if (r >= c->R) return -1;
    const size_t n = (size_t)c->L * c->L;
    const int32_t *h = c->h + (size_t)r * n;
    __int128 m[4] = { 0, 0, 0, 0 };
    for (size_t i = 0; i < n; ++i) {
        const __int128 d = (__int128)h[i] - (__int128)base;
        m[0] += d;
        m[1] += d * d;
        m[2] += d * d * d;
        m[3] += d * d * d * d;
    }
    for (int k = 0; k < 4; ++k) {
        out[2 * k] = (uint64_t)(unsigned __int128)m[k];
        out[2 * k + 1] = (uint64_t)((unsigned __int128)m[k] >> 64);
    }
    return 0;
}
