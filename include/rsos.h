/*
 * rsos.h -- C ABI of librsos: the B200 (sm_100a) hot path of the restricted solid-on-solid (RSOS)
 * deposition Monte Carlo of arXiv 1605.02620 (Kelling, Odor, Gemming).
 *
 * Citations:  P:n = /root/reference/PAPER.md line n;  D:x = DESIGN.md section x (the seeded
 * schedule DT(S,K) / RS restated from SURVEY.md 8(c).1, and the readings Q1..Q16 of the paper).
 *
 * What the library computes (Eq. 6): on a periodic L x L integer height lattice a site x
 * is picked at random and h(x) += 1 is accepted iff afterwards |h(x) - h(x')| <= N for the four
 * nearest neighbours x'.  R independent realizations are advanced at once; one Monte-Carlo
 * step (MCS) is L*L attempts per realization (reading Q4).  Large lattices are updated by
 * double tiling with a randomly moved origin: tiles of side S in four colour sets, one
 * seeded origin per sub-sweep, S*S/K sequential attempts per tile per sub-sweep (D:2).  All random
 * numbers come from Philox4x32-10 keyed by the seed with counter (call, tile, sub-sweep,
 * realization), so a realization is a pure function of (seed, r, L, N, S, K).  The squared
 * interface width W^2(L,t) (Eq. 2) is returned from exact integer sums.
 *
 * Conventions for every entry point
 *   - plain C, no exceptions; returns RSOS_OK (0) or a negative RSOS_E* code, and a failed call
 *     has no partial effect on the context (except after RSOS_ECUDA, when the context is dead);
 *   - rsos_last_error() returns a thread-local, NUL-terminated message for the last failure;
 *   - "host" pointers are ordinary CPU memory owned by the caller (pinned or pageable), "device"
 *     pointers are CUDA global memory of the context's device;
 *   - all work is enqueued on the context's stream; calls that return host data synchronise
 *     that stream before returning, rsos_advance does not;
 *   - a context is not thread-safe; distinct contexts are independent.
 * There is no CPU fallback: without a CUDA device every call fails with RSOS_ECUDA.
 */
#ifndef RSOS_H
#define RSOS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rsos_ctx rsos_ctx;

enum {
    RSOS_OK       =  0,
    RSOS_EINVAL   = -1,   /* bad argument (message says which)                                   */
    RSOS_ERANGE   = -2,   /* a counter would overflow: (t + mcs) * K >= 2^32, or sum h^2 >= 2^64 */
    RSOS_ENOMEM   = -3,   /* host or device allocation failed                                    */
    RSOS_ECUDA    = -4,   /* CUDA runtime error (message carries cudaGetErrorString)             */
    RSOS_EUNSUP   = -5    /* the requested engine cannot run this configuration                  */
};

/* Update engines.  All of them produce bit-identical heights (tests/test_gpu_parity.py).       */
enum {
    RSOS_ENGINE_AUTO   = 0,  /* RS mode: LEVEL for few realizations (R <= 2 x SM count), else     */
                             /* ONCHIP when the lattice fits in shared memory, else SIMPLE.       */
                             /* DT mode: FINE when it applies (tile 8 or 16, L <= 512), else      */
                             /* THREAD when it applies and one colour pass has at least           */
                             /* RSOS_THREAD_MIN_TILES active tiles, else RESIDENT when it         */
                             /* applies, else WARP, else SIMPLE.  L not a power of two: THREAD    */
                             /* (packed lattice, one lane per tile) under the condition stated    */
                             /* at rsos_init, else SIMPLE.                                        */
                             /* rsos_plan() tells what a given set of arguments selects.          */
    RSOS_ENGINE_SIMPLE = 1,  /* one thread per active tile, heights in global memory (slow;       */
                             /* the literal loop nest of D:2, kept as an on-device cross-check;   */
                             /* also the engine of the general-L schedule D:2b)                   */
    RSOS_ENGINE_WARP   = 2,  /* DT mode: one warp per active tile, (S+2)^2 window staged in       */
                             /* shared memory, 32 attempts in flight with exact conflict votes;   */
                             /* needs tile <= 128 and N <= 31                                     */
    RSOS_ENGINE_ONCHIP = 3,  /* RS mode (2S > L): one warp per realization, the whole lattice     */
                             /* stays in shared memory for all MCS of one rsos_advance call       */
    RSOS_ENGINE_THREAD = 4,  /* DT mode: one thread per active tile, the tile window held in      */
                             /* bank-interleaved shared memory at 2 (N = 1) or 4 (N <= 7) bits    */
                             /* per site; needs tile <= 64 and N <= 7                             */
    RSOS_ENGINE_FINE = 6,    /* DT mode with the paper's small sequential units ("domain sizes of 8 x 8  */
                             /* lattice sites", P:204 16 x 16): tile = 8 or 16, N <= 7, L <= 512.  One thread */
                             /* per cell works straight on a 4-bit lattice that stays in shared memory for    */
                             /* all passes of an rsos_advance call (one or more realizations per block)       */
    RSOS_ENGINE_MULTI = 7,   /* the schedule of opts.multisurface: one warp per 32 realizations that share    */
                             /* their coordinates, surfaces in shared memory with the realization innermost   */
                             /* (every access coalesced and conflict-free); serial mode, L <= 32, N <= 31     */
    RSOS_ENGINE_LEVEL = 8,   /* RS mode with few realizations (AUTO: R <= 2 x SM count): a block per          */
                             /* realization keeps the lattice in shared memory and runs batches of 512        */
                             /* consecutive attempts in dependency levels (an attempt waits only for earlier  */
                             /* attempts at equal or adjacent sites); 16 <= L <= 128                          */
    RSOS_ENGINE_RESIDENT = 5 /* DT mode, small lattices: a cluster of thread blocks keeps the     */
                             /* lattice of one realization in (distributed) shared memory for     */
                             /* every colour pass, sub-sweep and MCS of an rsos_advance call; one */
                             /* warp per tile, 32 attempts in flight with exact conflict votes.   */
                             /* Needs 16 <= tile <= 64, N <= 7 and the lattice in the shared      */
                             /* memory of at most 16 blocks (L <= 512 at N = 1)                   */
};
#define RSOS_THREAD_MIN_TILES 4096u

/* Options; all fields optional, zero = default.  Passed by pointer, copied by rsos_init.       */
typedef struct rsos_opts {
    uint32_t tile;        /* S: tile side, power of two >= 8; default 64.  2*S > L selects the    */
                          /* serial random-sequential mode RS (one tile = the lattice) (D:2)      */
    uint32_t subsweeps;   /* K: sub-sweeps per MCS, power of two, K | S*S, S*S/K >= 32; default 1 */
    uint32_t first_real;  /* global index of realization 0 (a run may be split over contexts)     */
    uint32_t engine;      /* RSOS_ENGINE_*                                                        */
    int32_t *d_heights;   /* DEVICE: borrowed buffer of R*L*L int32 (h[r][y][x], row-major, 16-   */
                          /* byte aligned), e.g. a torch tensor; NULL = the library allocates.    */
                          /* Its content on entry is ignored: rsos_init zeroes it (flat start).   */
                          /* With the THREAD, RESIDENT and FINE engines the working state is a    */
                          /* packed lattice (D:5) and this buffer is brought up to date only by   */
                          /* rsos_get_heights, rsos_moments, rsos_set_state, rsos_device_heights. */
    void    *stream;      /* cudaStream_t to enqueue on; NULL = the legacy default stream         */
    int32_t  device;      /* CUDA device ordinal + 1; 0 = the current device (so that a zeroed    */
                          /* struct means "all defaults"; SURVEY 8(b) wrote -1 = current instead)  */
    uint32_t lanes;       /* THREAD engine: lanes that share one tile, 1, 2, 4 or 8 (8 * lanes must not   */
                          /* exceed tile^2 / subsweeps); 0 = chosen from the number of tiles per colour   */
                          /* pass (D:4).  Does not change the result.                                     */
    uint32_t poisson;     /* 1: the Poisson variant DTP(c) of the schedule (D:2c): tile = 8 or 16,  */
                          /* K = tile^2 / 4 sub-sweeps per MCS (subsweeps must be 0 or that value), and in every   */
                          /* sub-sweep a cell makes n ~ Poisson(4) attempts instead of exactly 4.  Agrees with     */
                          /* serial dynamics where fixed counts on such small cells are 3.6 % low in W^2; the      */
                          /* number of attempts per MCS is L^2 on average only.  FINE engine (L <= 512, N <= 7).   */
    uint32_t cluster;     /* RESIDENT engine: thread blocks per realization (a thread-block cluster that  */
                          /* shares its shared memory), 1, 2, 4, 8 or 16; must divide the (L / 2 tile)^2  */
                          /* tiles of a colour pass; 0 = chosen by the library.  Does not change the      */
                          /* result.                                                                      */
    uint32_t multisurface;/* 1: the paper's shared-coordinate multisurface scheme (schedule MS, D:2d): groups */
                          /* of 128 realizations (by global index) share one coordinate sequence of 2 L^2           */
                          /* selections per MCS, and a member attempts a selection iff its own random bit is set    */
                          /* ("updating only half of the selected lattice sites"): L^2 attempts per surface and MCS  */
                          /* on average.  A different stochastic process from the default (surfaces of a group are  */
                          /* correlated); serial mode (2 * tile > L), L <= 32, N <= 31, first_real % 32 == 0.        */
} rsos_opts;

/*
 * rsos_init -- create a context: R flat surfaces h = 0 at t = 0, accepted = 0.
 *   ctx   out, host: receives the context (NULL on failure)
 *   L     lattice side, 4 <= L <= 65536 (periodic in both directions, reading Q2).  Powers of two run the
 *         schedule D:2 on every engine; any other L (the paper's L = 9605) runs the general-L schedule
 *         D:2b -- tiles of two sizes that divide the lattice, sites drawn by an exactly uniform bounded
 *         draw -- on the THREAD engine (packed lattice, one lane per tile) when tile = 64, N <= 7 and
 *         ceil(L / T) <= 66 with T = 2 floor(L / 128) (every L >= 4224, e.g. 9605), else on the SIMPLE engine
 *         (int32 heights; byte tile windows in shared memory when N <= 7)
 *   N     height-difference bound of Eq. (6), 1 <= N <= 127
 *   R     number of independent realizations, >= 1, R*L*L*4 bytes must fit on the device
 *   seed  Philox key (low word, high word)
 *   opts  host, may be NULL
 * Errors: RSOS_EINVAL (L, N, R, tile, subsweeps, engine, misaligned d_heights), RSOS_EUNSUP
 * (engine cannot run the mode; L not a power of two: engines other than AUTO, SIMPLE and -- under the
 * condition above -- THREAD),
 * RSOS_ENOMEM, RSOS_ECUDA.
 */
int rsos_init(rsos_ctx **ctx, uint32_t L, uint32_t N, uint32_t R, uint64_t seed, const rsos_opts *opts);

/*
 * rsos_advance -- advance every realization by `mcs` Monte-Carlo steps of the schedule D:2
 * (P:61-63 rule, P:77 decomposition): t += mcs.  Asynchronous: kernels are enqueued on the
 * context's stream and the call returns.  mcs = 0 is a no-op.  Contexts on different streams run concurrently:
 * when one context has few tiles per colour pass (BASELINE configs[1]: 8192), calling rsos_advance on several
 * contexts (one per seed, a stream each) before reading any of them back fills the GPU (D:11: 304 against 197 G
 * attempts/s for the four seeds of configs[1]).
 * Errors: RSOS_ERANGE if (t + mcs) * K >= 2^32 (nothing is enqueued), RSOS_ECUDA.
 */
int rsos_advance(rsos_ctx *ctx, uint64_t mcs);

/*
 * rsos_sums -- exact integer sums per realization (Eq. 2):
 *   S1[r] = sum_x h(x)  (int64),  S2[r] = sum_x h(x)^2  (uint64),  accepted[r] = accepted deposits.
 * Host buffers of R elements each; any of them may be NULL.  Synchronises the stream.
 * Errors: RSOS_ERANGE if max(h)^2 * L^2 could reach 2^64 (checked on the device), RSOS_ECUDA.
 */
int rsos_sums(rsos_ctx *ctx, int64_t *S1, uint64_t *S2, int64_t *accepted);

/*
 * rsos_width -- W2[r] = (L^2 * S2 - S1^2) / L^4 and hmean[r] = S1 / L^2 as doubles (Eq. 2), the
 * numerator formed exactly in 128-bit integers and converted once (L^4 is a power of two, so W2
 * is the correctly rounded exact value).  Host buffers of R doubles; either may be NULL.
 * Synchronises the stream.  Errors as rsos_sums.
 */
int rsos_width(rsos_ctx *ctx, double *W2, double *hmean);

/*
 * rsos_sums_static -- the sums of rsos_sums (Eq. 2) for code that is not allowed to allocate.
 *
 * Who this is for.  rsos_init obtains its reduction buffers with cudaMalloc, and some users of the width sums cannot
 * make that call, or any call that ends in it: an analysis step that runs inside a job whose device memory has been
 * handed over in full to another pool (a framework's caching allocator sized to the whole GPU leaves a raw cudaMalloc
 * nothing to take, so it fails), and a measurement loop that may not stall, because cudaMalloc and cudaFree wait for
 * the whole device and so serialise every stream of the process.  Such callers already own their buffers; this call
 * works entirely inside them plus one fixed array that belongs to the library.
 *
 * What it does.  d_heights holds R surfaces of L x L int32 heights on the CURRENT device (h[r][y][x], row-major; the
 * layout of rsos_device_heights, whose pointer may be passed straight in).  The call enqueues on `stream` the same
 * reduction kernel rsos_sums uses and writes, for r < R:
 *     d_S1[r]     = sum_x h(x)        (int64)
 *     d_S2[r]     = sum_x h(x)^2      (uint64, exact modulo 2^64)
 *     d_maxabs[r] = max_x |h(x)|      (uint32)
 * S2 is the true sum whenever maxabs^2 * L^2 < 2^64 (the condition rsos_sums turns into RSOS_ERANGE; here the caller
 * checks it, because reading the value back would force a synchronisation).  No context is needed, nothing is read
 * back to the host, and the call returns without waiting for the GPU.
 *
 *   d_heights  DEVICE, in: R*L*L int32, 16-byte aligned (4-byte if L*L is not a multiple of 4), not modified
 *   L          4 <= L <= 65536, any value
 *   R          1 <= R <= RSOS_STATIC_MAX_R; more is refused with RSOS_EINVAL and a message naming the limit
 *   d_S1, d_S2, d_maxabs   DEVICE, out: R elements each, caller-owned, any may be NULL (not all three)
 *   stream     cudaStream_t to enqueue on; NULL = the legacy default stream
 *
 * The fixed array.  The kernel accumulates with atomics into 32 bytes per realization.  For this call those bytes sit
 * in a file-scope __device__ array of RSOS_STATIC_MAX_R rows (128 KiB) compiled into librsos: every GPU on which the
 * library's code is loaded carries that array until the process exits, whether or not this function is ever called.
 * The call itself uses no cudaMalloc, cudaFree, cudaMallocHost or any routine that allocates.
 *   - First call on each device: the function looks up where that device keeps the array (cudaGetSymbolAddress, which
 *     may also make the runtime load the library's device code there) and remembers the answer; later calls on that
 *     device skip this.  Make this first call during start-up, with the intended device current, and before any
 *     stream capture is begun on that device.
 *   - The array is shared by all calls and keeps whatever the previous call left in it.  Each call therefore zeroes, on
 *     `stream`, exactly the rows it is about to use before the kernel adds into them; nothing else needs clearing.
 *   - Because of that sharing, two calls whose GPU work can overlap -- different streams, or two host threads -- add
 *     into the same rows and both get wrong sums.  Keep all calls for one device on one stream, or order them with
 *     events.  Calls on different devices do not interact.
 *
 * Errors: RSOS_EINVAL (NULL or misaligned pointer, L or R out of range -- nothing is enqueued), RSOS_ECUDA.
 */
#define RSOS_STATIC_MAX_R 4096u
int rsos_sums_static(const int32_t *d_heights, uint32_t L, uint32_t R, int64_t *d_S1, uint64_t *d_S2,
                     uint32_t *d_maxabs, void *stream);

/*
 * rsos_moments -- (Eq. 13-15) exact central power sums about the
 * integer base b[r] = floor(S1[r] / L^2):  M[r][k-1] = sum_x (h(x) - b[r])^k for k = 1..4 as
 * signed 128-bit integers stored little-endian in two uint64 words (lo, hi): out[r][k-1][2].
 * Host buffers: base (R int64, may be NULL) and out (R*4*2 uint64).  Synchronises the stream.
 */
int rsos_moments(rsos_ctx *ctx, int64_t *base, uint64_t *out);

/*
 * rsos_height_moments -- central moments of the height distribution of each surface (Eq. 13, P:180-184,
 * with the observable h(x) and the empirical distribution of the L*L sites of one realization):
 *   hbar[r] = (1/L^2) sum_x h(x),   phi[r][n-2] = (1/L^2) sum_x (h(x) - hbar[r])^n  for n = 2, 3, 4.
 * Formed on the host from the exact 128-bit power sums of rsos_moments (binomial expansion about the
 * integer base, extended precision), so the only rounding is the final conversion to double.  The
 * ensemble skewness / kurtosis of Eq. (14), (15) are <phi3> / <phi2>^(3/2) and <phi4> / <phi2>^2 - 3.
 * Host buffers: hbar (R doubles, may be NULL), phi (R*3 doubles).  Synchronises the stream.
 * Errors as rsos_moments.
 */
int rsos_height_moments(rsos_ctx *ctx, double *hbar, double *phi);

/*
 * rsos_get_heights -- copy realizations r0 .. r0+nr-1 (nr*L*L int32, h[r][y][x]) to host_out.
 * Synchronises the stream.  Errors: RSOS_EINVAL if the range is outside [0, R), RSOS_ECUDA.
 */
int rsos_get_heights(rsos_ctx *ctx, uint32_t r0, uint32_t nr, int32_t *host_out);

/*
 * rsos_set_state -- overwrite realizations r0 .. r0+nr-1 from host_in (same layout), set the sweep
 * counter t (applies to all realizations) and, if accepted != NULL, their accepted counters
 * (host, nr int64).  For snapshot restarts: t enters the Philox counter, so (heights, t) is the
 * whole state.  Synchronises the stream.  Every engine relies on Eq. (6), so the written surfaces
 * are checked on the device: if some bond has |dh| > N the call returns RSOS_EINVAL -- the one
 * failure WITH an effect: the realizations hold host_in and t is set, and the context is marked
 * invalid: rsos_advance, rsos_sums, rsos_width, rsos_moments and rsos_get_heights fail with
 * RSOS_EINVAL until a later rsos_set_state leaves every surface of the context valid (while the
 * mark is set, rsos_set_state checks the whole lattice, not only what it wrote).
 */
int rsos_set_state(rsos_ctx *ctx, uint32_t r0, uint32_t nr, const int32_t *host_in,
                   uint64_t t, const int64_t *accepted);

/* rsos_time -- *t = number of MCS done since the flat start (host pointer). */
int rsos_time(rsos_ctx *ctx, uint64_t *t);

/*
 * rsos_info -- describe the context: out[0] = mode (0 RS, 1 DT), out[1] = engine in use,
 * out[2] = S (effective tile side), out[3] = K, out[4] = kernel launches enqueued so far,
 * out[5] = device SM count, out[6] = shared-memory bytes per block of the update kernel,
 * out[7] = update-kernel blocks per launch, out[8] = lanes per tile (THREAD / RESIDENT, else 0),
 * out[9] = bits per site of the packed working lattice (THREAD / RESIDENT engine, else 0),
 * out[10] = RESIDENT engine blocks per cluster (else 0), out[11] = 1 if the int32 height buffer
 * exists (it is allocated on first use when the working state is the packed lattice).
 * Host buffer of 12 uint64.
 */
int rsos_info(rsos_ctx *ctx, uint64_t *out);

/*
 * rsos_device_heights -- *d = the DEVICE pointer of the int32 height buffer (borrowed or owned),
 * valid until rsos_free.  The call first brings the buffer up to date on the context's stream
 * (THREAD engine: rebuilt from the packed working lattice, D:5); its content is current as of this
 * call and goes stale with the next rsos_advance.  Reads must be ordered after the stream.
 */
int rsos_device_heights(rsos_ctx *ctx, int32_t **d);

/*
 * rsos_kernel_time -- accumulated device time of the update kernels, measured with CUDA events on
 * the context's stream when timing was enabled with enable != 0 (it then records two events
 * around the update launches of every rsos_advance; conversions between the packed and the int32
 * lattice and the width kernels lie outside them).  Synchronises the stream.  *ms_total and
 * *n_launches (host) receive the time and the number of update-kernel launches since timing was
 * enabled; enable = 0 switches it off.  Either pointer may be NULL.
 */
int rsos_kernel_time(rsos_ctx *ctx, int enable, double *ms_total, uint64_t *n_launches);

/*
 * rsos_plan -- what rsos_init would choose for (L, N, R, opts) on a device with sm_count SMs
 * (<= 0: the current CUDA device's count, or 148 -- a B200 -- when there is no device): pure host
 * logic, needs no CUDA device.  out (host, 9 uint64): out[0] = mode
 * (0 RS, 1 DT), out[1] = engine, out[2] = S, out[3] = K, out[4] = active tiles per colour pass
 * (0 in RS mode), out[5] = lanes per tile (THREAD / RESIDENT, else 0), out[6] = bits per site of the
 * packed lattice (else 0), out[7] = kernel launches per MCS (RS mode and RESIDENT: per call),
 * out[8] = RESIDENT engine blocks per cluster (else 0); out is 9 uint64.  Same argument errors as rsos_init.
 */
int rsos_plan(uint32_t L, uint32_t N, uint32_t R, const rsos_opts *opts, int sm_count, uint64_t *out);

/* rsos_free -- release the context and everything the library allocated (not d_heights). */
void rsos_free(rsos_ctx *ctx);

/* rsos_last_error -- message of the last failed call on this thread ("" if none). */
const char *rsos_last_error(void);

/*
 * rsos_philox -- test hook: Philox4x32-10 of n (counter, key) pairs evaluated ON THE DEVICE by the
 * same device function the update kernels use.  Host buffers: ctr (n*4 uint32), key (n*2 uint32),
 * out (n*4 uint32).  Used to cross-check the generator against the oracle's and cuRAND's.
 */
int rsos_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint32_t n);

#ifdef __cplusplus
}
#endif
#endif /* RSOS_H */
