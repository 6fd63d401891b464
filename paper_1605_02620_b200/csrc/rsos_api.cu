// rsos_api.cu -- the C ABI of librsos (include/rsos.h): argument checking, context, launch loops.
// Product code (CUDA path).  No CPU fallback: every compute step runs in the kernels of
// rsos_update.cu / rsos_reduce.cu.  Shares nothing with oracle/.
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/rsos.h"
#include "rsos_device.cuh"
#include "rsos_internal.h"

using namespace rsos;

struct rsos_ctx {
    Params p;
    bool mode_dt;
    uint32_t engine;
    uint64_t seed;
    uint64_t t;
    uint64_t launches;
    int device;
    cudaStream_t stream;
    bool own_heights;
    unsigned long long *d_red;        // R * 8 uint64 scratch for reductions
    unsigned long long *h_red;        // pinned mirror
    long long *d_base;                // R int64 (moments)
    int sm_count;
    uint32_t blocks;                  // update-kernel blocks per launch
    // THREAD engine: the working state is the packed lattice p.pk; the int32 heights p.h are rebuilt on demand
    bool h_valid, pk_valid;           // which of the two copies is current (both after init)
    long long *d_s1off;               // R int64: sum h = s1off + accepted while pk is the current copy
    int32_t *d_V;                     // R * L int32 scratch (column chain)
    unsigned long long *d_srel;       // 4R uint64 scratch (sum rel, sum rel^2, min rel, max rel)
    unsigned long long *h_pk;         // pinned host mirror: 4R (d_srel) + R (s1off) uint64
    int32_t *d_h00;                   // R int32 scratch
    size_t smem_bytes;
    // optional timing of rsos_advance
    bool timing;
    cudaEvent_t ev0, ev1;
    double ms_total;
    uint64_t timed_launches;
    uint64_t launches_at_ev0, launches_at_ev1;
    bool ev_pending;
    // set by a rsos_set_state that wrote a surface violating Eq. (6); cleared by a set_state after which the
    // whole lattice passes the check.  While set, every call that would run an engine or read sums fails.
    bool state_invalid;
};

static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                                   \
    do {                                                                                                 \
        cudaError_t e_ = (expr);                                                                         \
        if (e_ != cudaSuccess) return fail(RSOS_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_));         \
    } while (0)

static bool is_pow2(uint64_t v) { return v && !(v & (v - 1)); }
static uint32_t ilog2(uint64_t v) { uint32_t l = 0; while ((1ull << l) < v) ++l; return l; }

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (dev != prev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

extern "C" const char *rsos_last_error(void) { return g_err; }

static void destroy(rsos_ctx *c)
{
    if (!c) return;
    if (c->own_heights && c->p.h) cudaFree(c->p.h);
    if (c->p.accepted) cudaFree(c->p.accepted);
    if (c->p.err) cudaFree(c->p.err);
    if (c->d_red) cudaFree(c->d_red);
    if (c->h_red) cudaFreeHost(c->h_red);
    if (c->d_base) cudaFree(c->d_base);
    if (c->p.pk) cudaFree(c->p.pk);
    if (c->d_s1off) cudaFree(c->d_s1off);
    if (c->d_V) cudaFree(c->d_V);
    if (c->d_srel) cudaFree(c->d_srel);
    if (c->h_pk) cudaFreeHost(c->h_pk);
    if (c->d_h00) cudaFree(c->d_h00);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    delete c;
}

// Host-only planning: argument checks, mode, engine selection, lanes and packed-site width.
// Shared by rsos_init and rsos_plan; needs no device.
struct Plan {
    bool mode_dt, general;
    uint32_t engine, S, K, lanes, field_bits, cluster, T;
    uint64_t pass_tiles;
};

constexpr size_t SMEM_LIMIT_SM100 = 227u * 1024u;        // opt-in shared memory per block on sm_100a (rsos_plan without a device)

static int make_plan(uint32_t L, uint32_t N, uint32_t R, const rsos_opts &opt, int sm_count, size_t smem_limit, Plan *pl)
{
    if (L < 4 || L > 65536) return fail(RSOS_EINVAL, "L = %u must be in [4, 65536]", L);
    const bool general = !is_pow2(L);                      // general-L schedule RSG / DTG (D:2b)
    if (N < 1 || N > 127) return fail(RSOS_EINVAL, "N = %u must be in [1, 127]", N);
    if (R < 1) return fail(RSOS_EINVAL, "R must be >= 1");
    if (opt.lanes != 0 && opt.lanes != 1 && opt.lanes != 2 && opt.lanes != 4 && opt.lanes != 8)
        return fail(RSOS_EINVAL, "opts.lanes = %u must be 0, 1, 2, 4 or 8", opt.lanes);
    if (opt.cluster != 0 && opt.cluster != 1 && opt.cluster != 2 && opt.cluster != 4 && opt.cluster != 8 && opt.cluster != 16)
        return fail(RSOS_EINVAL, "opts.cluster = %u must be 0, 1, 2, 4, 8 or 16", opt.cluster);
    if (opt.engine > RSOS_ENGINE_LEVEL) return fail(RSOS_EINVAL, "unknown engine %u", opt.engine);
    uint32_t S = opt.tile ? opt.tile : 64, K = opt.subsweeps ? opt.subsweeps : 1;
    if (!is_pow2(S) || S < 8) return fail(RSOS_EINVAL, "tile = %u must be a power of two >= 8", S);
    if (opt.poisson > 1) return fail(RSOS_EINVAL, "opts.poisson = %u must be 0 or 1", opt.poisson);
    if (opt.multisurface > 1) return fail(RSOS_EINVAL, "opts.multisurface = %u must be 0 or 1", opt.multisurface);
    if (opt.multisurface && opt.poisson) return fail(RSOS_EINVAL, "opts.multisurface and opts.poisson exclude each other");
    if (opt.poisson) {                                     // D:2c: K = tile^2 / 4 sub-sweeps of Poisson(4) attempts per cell
        if (S != 8 && S != 16) return fail(RSOS_EINVAL, "opts.poisson needs tile = 8 or 16");
        if (opt.subsweeps && opt.subsweeps != S * S / 4) return fail(RSOS_EINVAL, "opts.poisson fixes subsweeps = tile^2 / 4 = %u", S * S / 4);
        K = S * S / 4;
    }
    if (!is_pow2(K)) return fail(RSOS_EINVAL, "subsweeps = %u must be a power of two", K);
    const bool mode_dt = 2ull * S <= L;
    if (mode_dt) {
        if (!opt.poisson && (((uint64_t)S * S) % K || (uint64_t)S * S / K < 32))
            return fail(RSOS_EINVAL, "subsweeps = %u must divide tile^2 with tile^2/subsweeps >= 32", K);
    } else {
        if (opt.poisson) return fail(RSOS_EINVAL, "opts.poisson needs DT mode (2 * tile <= L)");
        S = L; K = 1;
    }
    if ((uintptr_t)opt.d_heights & 15u) return fail(RSOS_EINVAL, "d_heights must be 16-byte aligned");
    if ((uint64_t)opt.first_real + R > 0xFFFFFFFFull) return fail(RSOS_EINVAL, "first_real + R overflows 32 bits");

    // engine selection (include/rsos.h)
    uint32_t engine = opt.engine;
    const bool warp_ok = !general && mode_dt && S <= 128 && N <= 31;
    const bool gthread_can = general && mode_dt && gthread_ok(L, N, S, K);      // general L on the packed lattice (S = 64)
    const bool thread_ok = (!general && mode_dt && S <= 64 && N <= 7) || gthread_can;
    const bool onchip_ok = !general && !mode_dt && L <= 128 && N <= 31;
    const uint32_t T = !mode_dt ? 0u : general ? 2u * (L / (2u * S)) : L / S;
    const uint64_t pass_tiles = mode_dt ? (uint64_t)R * (T / 2) * (T / 2) : 0;
    // RESIDENT: blocks per cluster (= per realization) = opts.cluster, else chosen from the shared memory a block
    // may use and the number of blocks the machine needs (rsos_resident.cu)
    uint32_t res_cluster = 0;
    if (mode_dt && !general) {
        if (opt.cluster) { if (resident_ok(L, N, S, K, opt.cluster, smem_limit)) res_cluster = opt.cluster; }
        else res_cluster = resident_cluster_size(L, N, S, K, R, sm_count, smem_limit);
    }
    if (opt.multisurface) {                                // D:2d: the shared-coordinate schedule MS, MULTI engine
        if (mode_dt || general) return fail(RSOS_EINVAL, "opts.multisurface needs the serial mode (2 * tile > L) on a power-of-two lattice");
        if (!multi_ok(L, N, opt.first_real))
            return fail(RSOS_EUNSUP, "opts.multisurface runs on the MULTI engine: L <= 32, N <= 31, first_real a multiple of 32");
        if (engine != RSOS_ENGINE_AUTO && engine != RSOS_ENGINE_MULTI) return fail(RSOS_EUNSUP, "opts.multisurface runs on the MULTI engine only");
        engine = RSOS_ENGINE_MULTI;
    } else if (engine == RSOS_ENGINE_MULTI) {
        return fail(RSOS_EINVAL, "engine MULTI runs the schedule of opts.multisurface only");
    }
    const bool fine_can = !general && mode_dt && fine_ok(L, N, S, K, opt.poisson != 0);
    if (opt.poisson && !fine_can)
        return fail(RSOS_EUNSUP, "opts.poisson runs on the FINE engine: L <= 512 (a power of two) and N <= 7");
    if (opt.poisson && engine != RSOS_ENGINE_AUTO && engine != RSOS_ENGINE_FINE)
        return fail(RSOS_EUNSUP, "opts.poisson runs on the FINE engine only");
    const bool level_can = !general && !mode_dt && !opt.multisurface && level_ok(L, N);
    if (engine == RSOS_ENGINE_AUTO) {
        // serial RS: a warp per realization (ONCHIP) when there are enough realizations to fill the machine, else a
        // block per realization that runs a batch of attempts in dependency levels (LEVEL)
        if (!mode_dt) engine = (level_can && R <= 2u * (uint32_t)sm_count) ? RSOS_ENGINE_LEVEL
                               : onchip_ok ? RSOS_ENGINE_ONCHIP : level_can ? RSOS_ENGINE_LEVEL : RSOS_ENGINE_SIMPLE;
        else if (fine_can) engine = RSOS_ENGINE_FINE;                  // 8- or 16-site cells on a lattice that fits on chip
        else if (thread_ok && pass_tiles >= RSOS_THREAD_MIN_TILES) engine = RSOS_ENGINE_THREAD;
        else if (res_cluster && pass_tiles / R <= 16) engine = RSOS_ENGINE_RESIDENT;   // few tiles per pass and realization
        else engine = warp_ok ? RSOS_ENGINE_WARP : thread_ok ? RSOS_ENGINE_THREAD : RSOS_ENGINE_SIMPLE;
    }
    if (engine == RSOS_ENGINE_RESIDENT && !res_cluster)
        return fail(RSOS_EUNSUP, "engine RESIDENT needs DT mode, 16 <= tile <= 64, N <= 7, a cluster size of 1, 2, 4, 8 or 16 that divides "
                                 "the (L / 2 tile)^2 tiles of a colour pass with at most 16 tiles per block, and the lattice slab in shared memory");
    if (engine == RSOS_ENGINE_FINE && !fine_can)
        return fail(RSOS_EUNSUP, "engine FINE needs DT mode with tile 8 or 16, N <= 7 and L <= 512 (the 4-bit lattice within 128 KiB)");
    if (engine == RSOS_ENGINE_LEVEL && !level_can)
        return fail(RSOS_EUNSUP, "engine LEVEL needs the serial mode (2 * tile > L), 16 <= L <= 128 (a power of two)");
    if (engine == RSOS_ENGINE_WARP && !warp_ok)
        return fail(RSOS_EUNSUP, "engine WARP needs DT mode (2*tile <= L), tile <= 128 and N <= 31");
    if (engine == RSOS_ENGINE_THREAD && !thread_ok)
        return fail(RSOS_EUNSUP, "engine THREAD needs DT mode (2*tile <= L), tile <= 64 and N <= 7");
    if (engine == RSOS_ENGINE_ONCHIP && !onchip_ok)
        return fail(RSOS_EUNSUP, "engine ONCHIP needs RS mode (2*tile > L), L <= 128 and N <= 31");
    if (general && engine != RSOS_ENGINE_SIMPLE && !(engine == RSOS_ENGINE_THREAD && gthread_can))
        return fail(RSOS_EUNSUP, "L = %u is not a power of two: the general-L schedule runs on the SIMPLE engine, and on the THREAD "
                                 "engine when tile = 64, N <= 7 and ceil(L / T) <= 66", L);
    pl->mode_dt = mode_dt; pl->general = general; pl->T = T;
    pl->engine = engine; pl->S = S; pl->K = K; pl->pass_tiles = pass_tiles;
    pl->lanes = 0; pl->field_bits = 0;
    pl->cluster = 0;
    if (engine == RSOS_ENGINE_RESIDENT) {
        pl->field_bits = thread_dt_field_bits(N, S);
        pl->lanes = 32;                                    // one warp per tile
        pl->cluster = res_cluster;
    }
    if (engine == RSOS_ENGINE_FINE) {
        pl->field_bits = thread_dt_field_bits(N, S);
        pl->lanes = 1;                                     // one thread per cell
    }
    if (engine == RSOS_ENGINE_THREAD) {
        pl->field_bits = thread_dt_field_bits(N, S);
        if (general && opt.lanes > 1) return fail(RSOS_EINVAL, "opts.lanes = %u: general L runs one lane per tile", opt.lanes);
        uint32_t kl = general ? 1u : opt.lanes ? opt.lanes : thread_dt_lanes_per_tile(pass_tiles, sm_count, pl->field_bits);
        while (!opt.lanes && 8ull * kl > (uint64_t)S * S / K) kl /= 2;                       // a batch is 8 * lanes attempts
        if (8ull * kl > (uint64_t)S * S / K)
            return fail(RSOS_EINVAL, "opts.lanes = %u needs tile^2 / subsweeps >= %u attempts per tile", kl, 8 * kl);
        pl->lanes = kl;
    }
    return RSOS_OK;
}

extern "C" int rsos_plan(uint32_t L, uint32_t N, uint32_t R, const rsos_opts *o, int sm_count, uint64_t *out)
{
    if (!out) return fail(RSOS_EINVAL, "out is NULL");
    rsos_opts opt;
    memset(&opt, 0, sizeof opt);
    if (o) opt = *o;
    Plan pl;
    if (sm_count <= 0) {                                   // the current device's SM count; 148 (a B200) without a device
        int dev = 0, smc = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&smc, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && smc > 0)
            sm_count = smc;
        else {
            cudaGetLastError();
            sm_count = 148;
        }
    }
    const int rc = make_plan(L, N, R, opt, sm_count, SMEM_LIMIT_SM100, &pl);
    if (rc) return rc;
    out[0] = pl.mode_dt ? 1 : 0; out[1] = pl.engine; out[2] = pl.S; out[3] = pl.K;
    out[4] = pl.pass_tiles; out[5] = pl.lanes; out[6] = pl.field_bits;
    out[7] = (pl.engine == RSOS_ENGINE_RESIDENT || pl.engine == RSOS_ENGINE_FINE) ? 1 : pl.mode_dt ? (uint64_t)4 * pl.K : 1;      // launches per MCS (RESIDENT, RS: per call)
    out[8] = pl.cluster;
    return RSOS_OK;
}

extern "C" int rsos_init(rsos_ctx **out, uint32_t L, uint32_t N, uint32_t R, uint64_t seed, const rsos_opts *o)
{
    if (!out) return fail(RSOS_EINVAL, "ctx is NULL");
    *out = nullptr;
    rsos_opts opt;
    memset(&opt, 0, sizeof opt);
    if (o) opt = *o;

    Plan pl;
    {   // argument errors are reported before any device is touched (the SM count only steers lanes per tile)
        const int rc0 = make_plan(L, N, R, opt, 1, SMEM_LIMIT_SM100, &pl);
        if (rc0) return rc0;
    }
    int dev = 0;
    if (opt.device > 0) dev = opt.device - 1;
    else CUDA_TRY(cudaGetDevice(&dev));
    DeviceGuard guard(dev);
    if (!guard.ok) return fail(RSOS_ECUDA, "cannot select CUDA device %d", dev);
    {
        int smc = 0, smem_optin = 0;
        CUDA_TRY(cudaDeviceGetAttribute(&smc, cudaDevAttrMultiProcessorCount, dev));
        CUDA_TRY(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        const int rc0 = make_plan(L, N, R, opt, smc, (size_t)smem_optin, &pl);
        if (rc0) return rc0;
    }
    const bool mode_dt = pl.mode_dt;
    const uint32_t engine = pl.engine, S = pl.S, K = pl.K;

    rsos_ctx *c = new (std::nothrow) rsos_ctx();
    if (!c) return fail(RSOS_ENOMEM, "out of host memory");
    memset(static_cast<void *>(c), 0, sizeof *c);
    c->device = dev;
    c->stream = (cudaStream_t)opt.stream;
    c->mode_dt = mode_dt;
    c->engine = engine;
    c->seed = seed;
    Params &p = c->p;
    p.L = L; p.lgL = ilog2(L); p.N = N; p.R = R; p.first_real = opt.first_real;
    p.S = S; p.lgS = ilog2(S); p.K = K;
    p.general = pl.general ? 1u : 0u; p.T = pl.T;
    p.poisson = opt.poisson ? 1u : 0u;
    p.multisurface = opt.multisurface ? 1u : 0u;
    p.k0 = (uint32_t)(seed & 0xFFFFFFFFull); p.k1 = (uint32_t)(seed >> 32);

#define INIT_TRY(expr, code)                                                                             \
    do {                                                                                                 \
        cudaError_t e_ = (expr);                                                                         \
        if (e_ != cudaSuccess) {                                                                         \
            const int rc_ = fail(e_ == cudaErrorMemoryAllocation ? RSOS_ENOMEM : (code), "%s: %s", #expr, \
                                 cudaGetErrorString(e_));                                                \
            if (e_ == cudaErrorMemoryAllocation) cudaGetLastError();                                     \
            destroy(c);                                                                                  \
            return rc_;                                                                                  \
        }                                                                                                \
    } while (0)

    const size_t bytes = (size_t)R * L * L * sizeof(int32_t);
    const bool packed_state = engine == RSOS_ENGINE_THREAD || engine == RSOS_ENGINE_RESIDENT || engine == RSOS_ENGINE_FINE;   // working state = packed lattice (D:5)
    if (opt.d_heights) { p.h = opt.d_heights; c->own_heights = false; }
    else if (!packed_state) { INIT_TRY(cudaMalloc(&p.h, bytes), RSOS_ECUDA); c->own_heights = true; }
    // else: the int32 heights are allocated by the first call that needs them (alloc_heights)
    INIT_TRY(cudaMalloc(&p.accepted, (size_t)R * sizeof(unsigned long long)), RSOS_ECUDA);
    INIT_TRY(cudaMalloc(&p.err, sizeof(uint32_t)), RSOS_ECUDA);
    INIT_TRY(cudaMalloc(&c->d_red, (size_t)R * 8 * sizeof(unsigned long long)), RSOS_ECUDA);
    INIT_TRY(cudaMallocHost(&c->h_red, (size_t)R * 8 * sizeof(unsigned long long)), RSOS_ECUDA);
    INIT_TRY(cudaMalloc(&c->d_base, (size_t)R * sizeof(long long)), RSOS_ECUDA);
    c->h_valid = c->pk_valid = true;
    if (packed_state) {
        p.FB = pl.field_bits;
        p.KL = pl.lanes;
        p.CS = pl.cluster;
        // FB bits per site; general L: rows of ceil(L * FB / 32) words
        const size_t pk_bytes = pl.general ? (size_t)R * L * ((L * p.FB + 31u) / 32u) * sizeof(uint32_t) : bytes / 32 * p.FB;
        INIT_TRY(cudaMalloc(&p.pk, pk_bytes), RSOS_ECUDA);
        INIT_TRY(cudaMalloc(&c->d_s1off, (size_t)R * sizeof(long long)), RSOS_ECUDA);
        INIT_TRY(cudaMalloc(&c->d_V, (size_t)R * L * sizeof(int32_t)), RSOS_ECUDA);
        INIT_TRY(cudaMalloc(&c->d_srel, (size_t)R * 4 * sizeof(unsigned long long)), RSOS_ECUDA);
        INIT_TRY(cudaMallocHost(&c->h_pk, (size_t)R * 5 * sizeof(unsigned long long)), RSOS_ECUDA);
        INIT_TRY(cudaMalloc(&c->d_h00, (size_t)R * sizeof(int32_t)), RSOS_ECUDA);
        INIT_TRY(cudaMemsetAsync(p.pk, 0, pk_bytes, c->stream), RSOS_ECUDA);                // flat start
        INIT_TRY(cudaMemsetAsync(c->d_s1off, 0, (size_t)R * sizeof(long long), c->stream), RSOS_ECUDA);
    }
    if (p.h) INIT_TRY(cudaMemsetAsync(p.h, 0, bytes, c->stream), RSOS_ECUDA);        // flat start
    else c->h_valid = false;
    INIT_TRY(cudaMemsetAsync(p.accepted, 0, (size_t)R * sizeof(unsigned long long), c->stream), RSOS_ECUDA);
    INIT_TRY(cudaMemsetAsync(p.err, 0, sizeof(uint32_t), c->stream), RSOS_ECUDA);
    INIT_TRY(cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev), RSOS_ECUDA);
    p.sm_count = (uint32_t)c->sm_count;
    INIT_TRY(configure_engine(p, engine, mode_dt), RSOS_ECUDA);
    c->blocks = engine_blocks(p, engine, mode_dt);
    INIT_TRY(cudaEventCreate(&c->ev0), RSOS_ECUDA);
    INIT_TRY(cudaEventCreate(&c->ev1), RSOS_ECUDA);
    c->smem_bytes = engine == RSOS_ENGINE_WARP ? warp_dt_smem(p.lgS) : engine == RSOS_ENGINE_ONCHIP ? warp_rs_smem(p.lgL)
                    : engine == RSOS_ENGINE_THREAD ? thread_dt_smem(p) : engine == RSOS_ENGINE_RESIDENT ? resident_smem(p)
                    : engine == RSOS_ENGINE_FINE ? fine_smem(p) : engine == RSOS_ENGINE_MULTI ? multi_smem(p)
                    : engine == RSOS_ENGINE_LEVEL ? level_smem(p) : 0;
#undef INIT_TRY
    *out = c;
    return RSOS_OK;
}

extern "C" void rsos_free(rsos_ctx *c)
{
    if (!c) return;
    DeviceGuard guard(c->device);
    cudaStreamSynchronize(c->stream);
    destroy(c);
}

static int flush_timing(rsos_ctx *c)
{
    if (c->timing && c->ev_pending) {
        CUDA_TRY(cudaEventSynchronize(c->ev1));
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, c->ev0, c->ev1));
        c->ms_total += ms;
        c->timed_launches += c->launches_at_ev1 - c->launches_at_ev0;
        c->ev_pending = false;
    }
    return RSOS_OK;
}

static int check_device_err(rsos_ctx *c)
{
    uint32_t e = 0;
    CUDA_TRY(cudaMemcpyAsync(&e, c->p.err, sizeof e, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    if (e) return fail(RSOS_ECUDA, "device-side consistency check failed (flags 0x%x)", e);
    return RSOS_OK;
}

// Packed working lattice (D:5): the int32 heights exist only once somebody asks for them.
static int alloc_heights(rsos_ctx *c)
{
    if (c->p.h) return RSOS_OK;
    const size_t bytes = (size_t)c->p.R * c->p.L * c->p.L * sizeof(int32_t);
    const cudaError_t e = cudaMalloc(&c->p.h, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        c->p.h = nullptr;
        return fail(e == cudaErrorMemoryAllocation ? RSOS_ENOMEM : RSOS_ECUDA, "int32 heights (%zu bytes): %s", bytes,
                    cudaGetErrorString(e));
    }
    c->own_heights = true;
    return RSOS_OK;
}

// THREAD engine: make the int32 heights current (packed lattice -> p.h, rsos_pack.cu).
static int ensure_heights(rsos_ctx *c)
{
    if (!c->p.pk || c->h_valid) return RSOS_OK;
    {
        const int rc = alloc_heights(c);
        if (rc) return rc;
    }
    uint32_t n = 0;
    CUDA_TRY(launch_unpack(c->p, c->d_s1off, c->d_V, c->d_srel, c->d_h00, c->stream, &n));
    c->launches += n;
    c->h_valid = true;
    return RSOS_OK;
}

// THREAD engine: make the packed lattice current (p.h -> packed, and s1off = sum h - accepted).
static int ensure_packed(rsos_ctx *c)
{
    if (!c->p.pk || c->pk_valid) return RSOS_OK;
    const Params &p = c->p;
    CUDA_TRY(launch_sums(p.h, p.L, p.R, c->d_red, c->sm_count, c->stream));
    CUDA_TRY(launch_s1off(p, c->d_red, c->d_s1off, c->stream));
    CUDA_TRY(launch_pack(p, c->stream));
    c->launches += (p.R + 65534) / 65535 + 2;
    c->pk_valid = true;
    return RSOS_OK;
}

extern "C" int rsos_advance(rsos_ctx *c, uint64_t mcs)
{
    if (!c) return fail(RSOS_EINVAL, "ctx is NULL");
    if (mcs == 0) return RSOS_OK;
    const Params &p = c->p;
    if (mcs >= (1ull << 32) || (c->t + mcs) * p.K >= (1ull << 32))
        return fail(RSOS_ERANGE, "(t + mcs) * K = (%llu + %llu) * %u reaches 2^32", (unsigned long long)c->t,
                    (unsigned long long)mcs, p.K);
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(RSOS_ECUDA, "cannot select CUDA device %d", c->device);
    if (c->state_invalid) return fail(RSOS_EINVAL, "the state violates Eq. (6) (last rsos_set_state); set a valid state first");
    if (c->p.pk) {
        const int rc = ensure_packed(c);
        if (rc) return rc;
        c->h_valid = false;
    }
    if (c->timing) {                                       // the events bracket the update launches only
        const int rc = flush_timing(c);
        if (rc) return rc;
        CUDA_TRY(cudaEventRecord(c->ev0, c->stream));
        c->launches_at_ev0 = c->launches;
    }
    if (c->engine == RSOS_ENGINE_RESIDENT || c->engine == RSOS_ENGINE_FINE) {
        // all colour passes and sub-sweeps of many MCS inside one launch; long calls are cut into launches of
        // about 2^36 attempts (a fraction of a second) so that the stream stays responsive
        const uint64_t per_mcs = (uint64_t)p.R * p.L * p.L;
        const uint64_t chunk = per_mcs >= (1ull << 36) ? 1 : (1ull << 36) / per_mcs;
        for (uint64_t m = 0; m < mcs; m += chunk) {
            const uint64_t n = mcs - m < chunk ? mcs - m : chunk;
            if (c->engine == RSOS_ENGINE_FINE) CUDA_TRY(fine_launch(p, (uint32_t)(c->t + m), (uint32_t)n, c->stream));
            else CUDA_TRY(resident_launch(p, (uint32_t)(c->t + m), (uint32_t)n, c->stream));
            ++c->launches;
        }
    } else if (c->mode_dt) {
        for (uint64_t m = 0; m < mcs; ++m)
            for (uint32_t k = 0; k < p.K; ++k) {
                const uint32_t u = (uint32_t)((c->t + m) * p.K + k);
                for (uint32_t colour = 0; colour < 4; ++colour) {
                    CUDA_TRY(launch_dt_pass(p, c->engine, u, colour, c->blocks, c->stream));
                    ++c->launches;
                }
            }
    } else if (c->engine == RSOS_ENGINE_MULTI) {
        for (uint64_t m = 0; m < mcs; m += 4096) {         // the on-chip int16 heights are good for 4096 MCS per launch
            const uint64_t n = mcs - m < 4096 ? mcs - m : 4096;
            CUDA_TRY(launch_rs_sweeps(p, c->engine, (uint32_t)(c->t + m), (uint32_t)n, c->blocks, c->stream));
            ++c->launches;
        }
    } else {
        CUDA_TRY(launch_rs_sweeps(p, c->engine, (uint32_t)c->t, (uint32_t)mcs, c->blocks, c->stream));
        ++c->launches;
    }
    if (c->timing) {
        CUDA_TRY(cudaEventRecord(c->ev1, c->stream));
        c->launches_at_ev1 = c->launches;
        c->ev_pending = true;
    }
    c->t += mcs;
    return RSOS_OK;
}


// THREAD engine, packed lattice current: S1, S2 and max |h| straight from the packed lattice
// (rsos_pack.cu): h = h00 + rel with h00 = (S1 - sum rel) / L^2 and S1 = s1off + accepted, so
// S2 = sum rel^2 + 2 h00 sum rel + L^2 h00^2.  All exact (128-bit on the host).
static int reduce_sums_packed(rsos_ctx *c)
{
    const Params &p = c->p;
    const size_t R = p.R;
    CUDA_TRY(launch_packed_sums(p, c->d_V, c->d_srel, c->stream));
    c->launches += 3;
    CUDA_TRY(cudaMemcpyAsync(c->h_pk, c->d_srel, R * 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaMemcpyAsync(c->h_pk + R * 4, c->d_s1off, R * sizeof(long long), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaMemcpyAsync(c->h_red + R * 4, p.accepted, R * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    const int rc = check_device_err(c);
    if (rc) return rc;
    const __int128 n = (__int128)p.L * p.L;
    for (size_t r = 0; r < R; ++r) {
        const long long srel = (long long)c->h_pk[4 * r], mn = (long long)c->h_pk[4 * r + 2], mx = (long long)c->h_pk[4 * r + 3];
        const unsigned long long srel2 = c->h_pk[4 * r + 1];
        const long long s1 = (long long)c->h_pk[4 * R + r] + (long long)c->h_red[4 * R + r];
        const long long num = s1 - srel;
        const long long n2 = (long long)p.L * p.L;
        const long long h00 = p.general ? num / n2 : num >> (2 * p.lgL);
        if (h00 * n2 != num)
            return fail(RSOS_ECUDA, "realization %zu: packed lattice is inconsistent with sum h (reconstruction not exact)", r);
        const long long lo = h00 + mn, hi = h00 + mx;
        const unsigned long long amax = (unsigned long long)((lo < 0 ? -lo : lo) > (hi < 0 ? -hi : hi) ? (lo < 0 ? -lo : lo)
                                                                                                     : (hi < 0 ? -hi : hi));
        const __int128 s2 = (__int128)srel2 + 2 * (__int128)h00 * srel + n * (__int128)h00 * h00;
        if (amax > 0x7FFFFFFFull || s2 < 0 || (s2 >> 64) != 0)
            return fail(RSOS_ERANGE, "realization %zu: max|h| = %llu makes sum h^2 overflow 64 bits", r, amax);
        c->h_red[4 * r] = (unsigned long long)s1;
        c->h_red[4 * r + 1] = (unsigned long long)s2;
        c->h_red[4 * r + 2] = amax;
    }
    return RSOS_OK;
}

static int reduce_sums(rsos_ctx *c)
{
    const Params &p = c->p;
    if (c->state_invalid) return fail(RSOS_EINVAL, "the state violates Eq. (6) (last rsos_set_state); set a valid state first");
    if (p.pk && !c->h_valid) {
        const int rc0 = reduce_sums_packed(c);
        if (rc0) return rc0;
    } else {
        CUDA_TRY(launch_sums(p.h, p.L, p.R, c->d_red, c->sm_count, c->stream));
        c->launches += (p.R + 65534) / 65535;
        CUDA_TRY(cudaMemcpyAsync(c->h_red, c->d_red, (size_t)p.R * 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost,
                                 c->stream));
        CUDA_TRY(cudaMemcpyAsync(c->h_red + (size_t)p.R * 4, p.accepted, (size_t)p.R * sizeof(unsigned long long),
                                 cudaMemcpyDeviceToHost, c->stream));
        const int rc = check_device_err(c);
        if (rc) return rc;
    }
    // sum h^2 must stay below 2^64: max|h|^2 * L^2 < 2^64
    for (uint32_t r = 0; r < p.R; ++r) {
        const unsigned __int128 mx = c->h_red[4 * (size_t)r + 2];
        if (mx * mx * ((unsigned __int128)p.L * p.L) >> 64)
            return fail(RSOS_ERANGE, "realization %u: max|h| = %llu makes sum h^2 overflow 64 bits", r,
                        (unsigned long long)mx);
    }
    return RSOS_OK;
}

extern "C" int rsos_sums(rsos_ctx *c, int64_t *S1, uint64_t *S2, int64_t *accepted)
{
    if (!c) return fail(RSOS_EINVAL, "ctx is NULL");
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(RSOS_ECUDA, "cannot select CUDA device %d", c->device);
    const int rc = reduce_sums(c);
    if (rc) return rc;
    const uint32_t R = c->p.R;
    for (uint32_t r = 0; r < R; ++r) {
        if (S1) S1[r] = (int64_t)c->h_red[4 * (size_t)r];
        if (S2) S2[r] = c->h_red[4 * (size_t)r + 1];
        if (accepted) accepted[r] = (int64_t)c->h_red[4 * (size_t)R + r];
    }
    return RSOS_OK;
}

// Context-free and allocation-free: see include/rsos.h.  Argument checks here, the work in rsos_reduce.cu.
extern "C" int rsos_sums_static(const int32_t *d_heights, uint32_t L, uint32_t R, int64_t *d_S1, uint64_t *d_S2,
                                uint32_t *d_maxabs, void *stream)
{
    if (!d_heights) return fail(RSOS_EINVAL, "d_heights is NULL");
    if (L < 4 || L > 65536) return fail(RSOS_EINVAL, "L = %u must be in [4, 65536]", L);
    if (R < 1) return fail(RSOS_EINVAL, "R must be >= 1");
    if (R > RSOS_STATIC_MAX_R)
        return fail(RSOS_EINVAL, "R = %u exceeds RSOS_STATIC_MAX_R = %u, the number of realizations the library's fixed scratch "
                                 "array holds: split the surfaces over several calls, or use rsos_sums on a context", R,
                    RSOS_STATIC_MAX_R);
    if (!d_S1 && !d_S2 && !d_maxabs) return fail(RSOS_EINVAL, "d_S1, d_S2 and d_maxabs are all NULL: nothing to write");
    const bool vec = ((uint64_t)L * L) % 4 == 0;
    if ((uintptr_t)d_heights & (vec ? 15u : 3u)) return fail(RSOS_EINVAL, "d_heights must be %u-byte aligned", vec ? 16u : 4u);
    if (((uintptr_t)d_S1 & 7u) || ((uintptr_t)d_S2 & 7u) || ((uintptr_t)d_maxabs & 3u))
        return fail(RSOS_EINVAL, "d_S1 / d_S2 must be 8-byte aligned and d_maxabs 4-byte aligned");
    CUDA_TRY(launch_sums_static(d_heights, L, R, reinterpret_cast<long long *>(d_S1), reinterpret_cast<unsigned long long *>(d_S2),
                                d_maxabs, static_cast<cudaStream_t>(stream)));
    return RSOS_OK;
}

extern "C" int rsos_width(rsos_ctx *c, double *W2, double *hmean)
{
    if (!c) return fail(RSOS_EINVAL, "ctx is NULL");
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(RSOS_ECUDA, "cannot select CUDA device %d", c->device);
    const int rc = reduce_sums(c);
    if (rc) return rc;
    const uint32_t R = c->p.R;
    const unsigned __int128 n = (unsigned __int128)c->p.L * c->p.L;
    const double nd = (double)c->p.L * (double)c->p.L;
    for (uint32_t r = 0; r < R; ++r) {
        const int64_t s1 = (int64_t)c->h_red[4 * (size_t)r];
        const uint64_t s2 = c->h_red[4 * (size_t)r + 1];
        const unsigned __int128 a1 = (unsigned __int128)(s1 < 0 ? -(__int128)s1 : (__int128)s1);
        const unsigned __int128 num = n * s2 - a1 * a1;              // >= 0 (Cauchy-Schwarz)
        if (W2) W2[r] = (double)num / (nd * nd);
        if (hmean) hmean[r] = (double)s1 / nd;
    }
    return RSOS_OK;
}

extern "C" int rsos_moments(rsos_ctx *c, int64_t *base, uint64_t *out)
{
    if (!c) return fail(RSOS_EINVAL, "ctx is NULL");
    if (!out) return fail(RSOS_EINVAL, "out is NULL");
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(RSOS_ECUDA, "cannot select CUDA device %d", c->device);
    if (c->state_invalid) return fail(RSOS_EINVAL, "the state violates Eq. (6) (last rsos_set_state); set a valid state first");
    int rc = ensure_heights(c);                            // the moment kernel reads the int32 heights
    if (rc) return rc;
    rc = reduce_sums(c);
    if (rc) return rc;
    const Params &p = c->p;
    long long *hb = reinterpret_cast<long long *>(c->h_red + (size_t)p.R * 5);
    for (uint32_t r = 0; r < p.R; ++r) {
        const int64_t s1 = (int64_t)c->h_red[4 * (size_t)r];
        const int64_t n2 = (int64_t)p.L * p.L;
        hb[r] = s1 >= 0 ? s1 / n2 : -((-s1 + n2 - 1) / n2);         // floor(S1 / L^2)
        if (base) base[r] = hb[r];
    }
    CUDA_TRY(cudaMemcpyAsync(c->d_base, hb, (size_t)p.R * sizeof(long long), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(launch_moments(p.h, p.L, p.R, c->d_base, c->d_red, c->sm_count, c->stream));
    c->launches += (p.R + 65534) / 65535;
    CUDA_TRY(cudaMemcpyAsync(out, c->d_red, (size_t)p.R * 8 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return RSOS_OK;
}

extern "C" int rsos_height_moments(rsos_ctx *c, double *hbar, double *phi)
{
    if (!c) return fail(RSOS_EINVAL, "ctx is NULL");
    if (!phi) return fail(RSOS_EINVAL, "phi is NULL");
    const uint32_t R = c->p.R;
    uint64_t *raw = static_cast<uint64_t *>(malloc((size_t)R * 8 * sizeof(uint64_t)));
    int64_t *base = static_cast<int64_t *>(malloc((size_t)R * sizeof(int64_t)));
    if (!raw || !base) { free(raw); free(base); return fail(RSOS_ENOMEM, "out of host memory"); }
    const int rc = rsos_moments(c, base, raw);
    if (rc == RSOS_OK) {
        const long double n = (long double)c->p.L * (long double)c->p.L;
        for (uint32_t r = 0; r < R; ++r) {
            long double a[4];
            for (int k = 0; k < 4; ++k) {
                const unsigned __int128 u = ((unsigned __int128)raw[8 * (size_t)r + 2 * k + 1] << 64) | raw[8 * (size_t)r + 2 * k];
                a[k] = (long double)(__int128)u / n;       // raw moment about the integer base, per site
            }
            const long double m1 = a[0];                   // 0 <= m1 < 1: the base is floor(mean)
            phi[3 * (size_t)r + 0] = (double)(a[1] - m1 * m1);
            phi[3 * (size_t)r + 1] = (double)(a[2] - 3 * m1 * a[1] + 2 * m1 * m1 * m1);
            phi[3 * (size_t)r + 2] = (double)(a[3] - 4 * m1 * a[2] + 6 * m1 * m1 * a[1] - 3 * m1 * m1 * m1 * m1);
            if (hbar) hbar[r] = (double)((long double)base[r] + m1);
        }
    }
    free(raw);
    free(base);
    return rc;
}

extern "C" int rsos_get_heights(rsos_ctx *c, uint32_t r0, uint32_t nr, int32_t *host_out)
{
    if (!c) return fail(RSOS_EINVAL, "ctx is NULL");
    if ((uint64_t)r0 + nr > c->p.R) return fail(RSOS_EINVAL, "realizations [%u, %u) outside [0, %u)", r0, r0 + nr, c->p.R);
    if (nr && !host_out) return fail(RSOS_EINVAL, "host_out is NULL");
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(RSOS_ECUDA, "cannot select CUDA device %d", c->device);
    if (c->state_invalid) return fail(RSOS_EINVAL, "the state violates Eq. (6) (last rsos_set_state); set a valid state first");
    {
        const int rc0 = ensure_heights(c);
        if (rc0) return rc0;
    }
    const size_t per = (size_t)c->p.L * c->p.L;
    if (nr) CUDA_TRY(cudaMemcpyAsync(host_out, c->p.h + r0 * per, nr * per * sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
    return check_device_err(c);
}

extern "C" int rsos_set_state(rsos_ctx *c, uint32_t r0, uint32_t nr, const int32_t *host_in, uint64_t t,
                              const int64_t *accepted)
{
    if (!c) return fail(RSOS_EINVAL, "ctx is NULL");
    if ((uint64_t)r0 + nr > c->p.R) return fail(RSOS_EINVAL, "realizations [%u, %u) outside [0, %u)", r0, r0 + nr, c->p.R);
    if (nr && !host_in) return fail(RSOS_EINVAL, "host_in is NULL");
    if (t * c->p.K >= (1ull << 32)) return fail(RSOS_ERANGE, "t * K reaches 2^32");
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(RSOS_ECUDA, "cannot select CUDA device %d", c->device);
    if (c->p.pk) {
        // realizations outside [r0, r0+nr) keep their state: bring the int32 copy up to date first.  When the whole
        // lattice is overwritten (or already invalid) there is nothing to keep.
        if (nr == c->p.R || c->state_invalid) {
            const int rc0 = alloc_heights(c);
            if (rc0) return rc0;
        } else {
            int rc0 = ensure_heights(c);
            if (rc0) return rc0;
            rc0 = check_device_err(c);                     // a failed reconstruction must not be handed on
            if (rc0) return rc0;
        }
        c->h_valid = true;
        c->pk_valid = false;
    }
    const size_t per = (size_t)c->p.L * c->p.L;
    if (nr) CUDA_TRY(cudaMemcpyAsync(c->p.h + r0 * per, host_in, nr * per * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream));
    if (nr && accepted)
        CUDA_TRY(cudaMemcpyAsync(c->p.accepted + r0, accepted, nr * sizeof(int64_t), cudaMemcpyHostToDevice, c->stream));
    c->t = t;
    // Every engine relies on Eq. (6): check what was written -- and, while an earlier call left an invalid
    // state behind, the whole lattice, so that the flag is only cleared when every surface is valid.
    const uint32_t c0 = c->state_invalid ? 0u : r0, cn = c->state_invalid ? c->p.R : nr;
    if (cn) {
        CUDA_TRY(launch_violations(c->p.h + c0 * per, c->p.L, c->p.lgL, cn, c->p.N, c->d_red, c->stream));
        ++c->launches;
        CUDA_TRY(cudaMemcpyAsync(c->h_red, c->d_red, sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    }
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    if (cn && c->h_red[0]) {
        c->state_invalid = true;
        return fail(RSOS_EINVAL, "the written state violates Eq. (6) on %llu bonds (|dh| > N = %u); set a valid state before advancing",
                    c->h_red[0], c->p.N);
    }
    c->state_invalid = false;
    return RSOS_OK;
}

extern "C" int rsos_time(rsos_ctx *c, uint64_t *t)
{
    if (!c || !t) return fail(RSOS_EINVAL, "NULL argument");
    *t = c->t;
    return RSOS_OK;
}

extern "C" int rsos_info(rsos_ctx *c, uint64_t *out)
{
    if (!c || !out) return fail(RSOS_EINVAL, "NULL argument");
    out[0] = c->mode_dt ? 1 : 0;
    out[1] = c->engine;
    out[2] = c->p.S;
    out[3] = c->p.K;
    out[4] = c->launches;
    out[5] = (uint64_t)c->sm_count;
    out[6] = c->smem_bytes;
    out[7] = c->blocks;
    out[8] = c->p.pk ? c->p.KL : 0;
    out[9] = c->p.pk ? c->p.FB : 0;
    out[10] = c->engine == RSOS_ENGINE_RESIDENT ? c->p.CS : 0;
    out[11] = c->p.h ? 1 : 0;
    return RSOS_OK;
}

extern "C" int rsos_device_heights(rsos_ctx *c, int32_t **d)
{
    if (!c || !d) return fail(RSOS_EINVAL, "NULL argument");
    {
        DeviceGuard guard(c->device);
        if (!guard.ok) return fail(RSOS_ECUDA, "cannot select CUDA device %d", c->device);
        int rc0 = alloc_heights(c);
        if (rc0) return rc0;
        rc0 = ensure_heights(c);
        if (rc0) return rc0;
        rc0 = check_device_err(c);                         // a failed reconstruction must not be handed out
        if (rc0) return rc0;
    }
    *d = c->p.h;
    return RSOS_OK;
}

extern "C" int rsos_kernel_time(rsos_ctx *c, int enable, double *ms_total, uint64_t *n_launches)
{
    if (!c) return fail(RSOS_EINVAL, "ctx is NULL");
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(RSOS_ECUDA, "cannot select CUDA device %d", c->device);
    const int rc = flush_timing(c);
    if (rc) return rc;
    if (ms_total) *ms_total = c->ms_total;
    if (n_launches) *n_launches = c->timed_launches;
    if (enable && !c->timing) { c->timing = true; c->ms_total = 0; c->timed_launches = 0; c->ev_pending = false; }
    if (!enable) c->timing = false;
    return RSOS_OK;
}

extern "C" int rsos_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint32_t n)
{
    if (n == 0) return RSOS_OK;
    if (!ctr || !key || !out) return fail(RSOS_EINVAL, "NULL argument");
    uint32_t *d = nullptr;
    CUDA_TRY(cudaMalloc(&d, (size_t)n * 10 * sizeof(uint32_t)));
    cudaError_t e = cudaMemcpy(d, ctr, (size_t)n * 4 * sizeof(uint32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d + (size_t)n * 4, key, (size_t)n * 2 * sizeof(uint32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = launch_philox(d, d + (size_t)n * 4, d + (size_t)n * 6, n, nullptr);
    if (e == cudaSuccess) e = cudaMemcpy(out, d + (size_t)n * 6, (size_t)n * 4 * sizeof(uint32_t), cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return fail(RSOS_ECUDA, "rsos_philox: %s", cudaGetErrorString(e));
    return RSOS_OK;
}
