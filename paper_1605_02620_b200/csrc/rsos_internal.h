// rsos_internal.h -- host-side declarations shared by the translation units of librsos.
// Product code (CUDA path).  Not part of the public ABI (that is include/rsos.h).
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

namespace rsos {

struct Params;

constexpr int WARP_DT_WARPS = 1;     // warps (= tiles) per block of the DT warp engine (1: even spread over SMs)
constexpr int WARP_RS_WARPS = 4;     // warps (= realizations) per block of the on-chip RS engine

enum : uint32_t { ENGINE_AUTO = 0, ENGINE_SIMPLE = 1, ENGINE_WARP = 2, ENGINE_ONCHIP = 3, ENGINE_THREAD = 4, ENGINE_RESIDENT = 5, ENGINE_FINE = 6, ENGINE_MULTI = 7, ENGINE_LEVEL = 8 };

// rsos_update.cu
size_t warp_dt_smem(uint32_t lgS);
size_t warp_rs_smem(uint32_t lgL);
cudaError_t configure_engine(const Params &p, uint32_t engine, bool mode_dt);
uint32_t engine_blocks(const Params &p, uint32_t engine, bool mode_dt);
cudaError_t launch_dt_pass(const Params &p, uint32_t engine, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st);
cudaError_t launch_rs_sweeps(const Params &p, uint32_t engine, uint32_t t0, uint32_t mcs, uint32_t blocks, cudaStream_t st);
cudaError_t launch_philox(const uint32_t *d_ctr, const uint32_t *d_key, uint32_t *d_out, uint32_t n, cudaStream_t st);

// rsos_thread.cu (lane-per-tile DT engine on the packed lattice)
uint32_t thread_dt_field_bits(uint32_t N, uint32_t S);
uint32_t thread_dt_lanes_per_tile(uint64_t pass_tiles, int sm_count, uint32_t field_bits);
size_t thread_dt_smem(const Params &p);
cudaError_t thread_dt_configure(const Params &p);
uint32_t thread_dt_blocks(const Params &p);
cudaError_t thread_dt_launch(const Params &p, uint32_t u, uint32_t colour, uint32_t blocks, cudaStream_t st);

// rsos_gthread.cu (lane-per-tile DT engine on the packed lattice for lattice sides that are not powers of two)
bool gthread_ok(uint32_t L, uint32_t N, uint32_t S, uint32_t K);
size_t gthread_smem(const Params &p);
uint32_t gthread_blocks(const Params &p);
cudaError_t gthread_configure(const Params &p);
cudaError_t gthread_launch(const Params &p, uint32_t u, uint32_t colour, cudaStream_t st);

// rsos_resident.cu (DT schedule with the packed lattice resident in shared memory for a whole rsos_advance)
bool resident_ok(uint32_t L, uint32_t N, uint32_t S, uint32_t K, uint32_t csize, size_t smem_limit);
uint32_t resident_cluster_size(uint32_t L, uint32_t N, uint32_t S, uint32_t K, uint32_t R, int sm_count, size_t smem_limit);
size_t resident_smem(const Params &p);
cudaError_t resident_configure(const Params &p);
uint32_t resident_blocks(const Params &p);
cudaError_t resident_launch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st);

// rsos_fine.cu (DT schedule with 8- or 16-site cells, thread per cell, lattice resident in shared memory)
bool fine_ok(uint32_t L, uint32_t N, uint32_t S, uint32_t K, bool poisson);
size_t fine_smem(const Params &p);
uint32_t fine_blocks(const Params &p);
cudaError_t fine_configure(const Params &p);
cudaError_t fine_launch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st);

// rsos_multi.cu (shared-coordinate multisurface schedule MS, realizations innermost in shared memory)
bool multi_ok(uint32_t L, uint32_t N, uint32_t first_real);
size_t multi_smem(const Params &p);
uint32_t multi_blocks(const Params &p);
cudaError_t multi_configure(const Params &p);
cudaError_t multi_launch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st);

// rsos_level.cu (serial RS of few realizations: a block per realization, a batch of attempts run in dependency levels)
bool level_ok(uint32_t L, uint32_t N);
size_t level_smem(const Params &p);
uint32_t level_blocks(const Params &p);
cudaError_t level_configure(const Params &p);
cudaError_t level_launch(const Params &p, uint32_t t0, uint32_t mcs, cudaStream_t st);

// rsos_pack.cu (packed working lattice <-> int32 heights)
cudaError_t launch_pack(const Params &p, cudaStream_t st);
cudaError_t launch_s1off(const Params &p, const unsigned long long *d_red, long long *d_s1off, cudaStream_t st);
cudaError_t launch_packed_sums(const Params &p, int32_t *d_V, unsigned long long *d_srel, cudaStream_t st);
cudaError_t launch_unpack(const Params &p, const long long *d_s1off, int32_t *d_V, unsigned long long *d_srel,
                          int32_t *d_h00, cudaStream_t st, uint32_t *launches);

// rsos_reduce.cu
// out: per realization 4 x uint64: S1 (as int64 bits), S2, max |h| (max over threads), unused
cudaError_t launch_sums(const int32_t *h, uint32_t L, uint32_t R, unsigned long long *d_out, int sm_count, cudaStream_t st);
// number of nearest-neighbour bonds with |dh| > N in nr surfaces (Eq. 6), added into *d_bad
cudaError_t launch_violations(const int32_t *h, uint32_t L, uint32_t lgL, uint32_t nr, uint32_t N, unsigned long long *d_bad,
                              cudaStream_t st);
// out: per realization 8 x uint64: M1..M4 as (lo, hi) two's-complement 128-bit
cudaError_t launch_moments(const int32_t *h, uint32_t L, uint32_t R, const long long *d_base,
                           unsigned long long *d_out, int sm_count, cudaStream_t st);
// rsos_sums_static: launch_sums into the library's fixed device array (no allocation), results copied to the three
// caller-owned device arrays (any of them may be null); R <= RSOS_STATIC_MAX_R, current device, enqueued on st
cudaError_t launch_sums_static(const int32_t *h, uint32_t L, uint32_t R, long long *d_S1, unsigned long long *d_S2,
                               unsigned int *d_maxabs, cudaStream_t st);

}  // namespace rsos
