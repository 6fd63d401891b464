"""paper_1605_02620_b200 -- B200 (sm_100a) hot path of the RSOS deposition Monte Carlo of
arXiv 1605.02620: CUDA kernels behind the C ABI of include/rsos.h plus a thin ctypes binding.
See DESIGN.md.  This package never imports oracle/ (the CPU oracle is test infrastructure)."""
from .binding import (ENGINE_AUTO, ENGINE_FINE, ENGINE_LEVEL, ENGINE_MULTI, ENGINE_ONCHIP, ENGINE_RESIDENT, ENGINE_SIMPLE, ENGINE_THREAD, ENGINE_WARP, LIB_PATH, SYMBOLS,  # noqa: F401
                      Rsos, RsosError, STATIC_MAX_R, load, philox, plan, sums_static)
