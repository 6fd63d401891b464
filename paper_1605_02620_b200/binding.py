"""Thin ctypes binding of librsos (include/rsos.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; nothing here computes.
There is no CPU fallback: if librsos.so is missing or no CUDA device is present the calls raise.
This module imports nothing from oracle/.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librsos.so")

ENGINE_AUTO, ENGINE_SIMPLE, ENGINE_WARP, ENGINE_ONCHIP, ENGINE_THREAD, ENGINE_RESIDENT, ENGINE_FINE, ENGINE_MULTI, ENGINE_LEVEL = 0, 1, 2, 3, 4, 5, 6, 7, 8
ENGINE_NAMES = {0: "auto", 1: "simple", 2: "warp", 3: "onchip", 4: "thread", 5: "resident", 6: "fine", 7: "multi", 8: "level"}
RSOS_OK, RSOS_EINVAL, RSOS_ERANGE, RSOS_ENOMEM, RSOS_ECUDA, RSOS_EUNSUP = 0, -1, -2, -3, -4, -5

# every symbol include/rsos.h declares (tests check the .so exports exactly these)
SYMBOLS = ("rsos_init", "rsos_advance", "rsos_sums", "rsos_width", "rsos_moments", "rsos_height_moments", "rsos_get_heights",
           "rsos_set_state", "rsos_time", "rsos_info", "rsos_device_heights", "rsos_kernel_time",
           "rsos_free", "rsos_last_error", "rsos_philox", "rsos_plan", "rsos_sums_static")
STATIC_MAX_R = 4096                # RSOS_STATIC_MAX_R of include/rsos.h


class RsosOpts(C.Structure):
    _fields_ = [("tile", C.c_uint32), ("subsweeps", C.c_uint32), ("first_real", C.c_uint32),
                ("engine", C.c_uint32), ("d_heights", C.c_void_p), ("stream", C.c_void_p),
                ("device", C.c_int32), ("lanes", C.c_uint32), ("poisson", C.c_uint32), ("cluster", C.c_uint32), ("multisurface", C.c_uint32)]


class RsosError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("librsos error %d: %s" % (code, msg))
        self.code = code


_lib = None


def load():
    """dlopen librsos.so (built by paper_1605_02620_b200.build) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RsosError(RSOS_ECUDA, "librsos.so not built: run `python -m paper_1605_02620_b200.build`")
    l = C.CDLL(LIB_PATH)
    u32, u64, vp, ci = C.c_uint32, C.c_uint64, C.c_void_p, C.c_int
    l.rsos_init.argtypes = [C.POINTER(vp), u32, u32, u32, u64, C.POINTER(RsosOpts)]
    l.rsos_advance.argtypes = [vp, u64]
    l.rsos_sums.argtypes = [vp, vp, vp, vp]
    l.rsos_width.argtypes = [vp, vp, vp]
    l.rsos_moments.argtypes = [vp, vp, vp]
    l.rsos_height_moments.argtypes = [vp, vp, vp]
    l.rsos_get_heights.argtypes = [vp, u32, u32, vp]
    l.rsos_set_state.argtypes = [vp, u32, u32, vp, u64, vp]
    l.rsos_time.argtypes = [vp, C.POINTER(u64)]
    l.rsos_info.argtypes = [vp, C.POINTER(u64)]
    l.rsos_device_heights.argtypes = [vp, C.POINTER(vp)]
    l.rsos_kernel_time.argtypes = [vp, ci, C.POINTER(C.c_double), C.POINTER(u64)]
    l.rsos_philox.argtypes = [vp, vp, vp, u32]
    l.rsos_sums_static.argtypes = [vp, u32, u32, vp, vp, vp, vp]
    for name in SYMBOLS:
        getattr(l, name).restype = ci
    l.rsos_free.restype = None
    l.rsos_last_error.restype = C.c_char_p
    _lib = l
    return l


def _check(rc):
    if rc != 0:
        raise RsosError(rc, load().rsos_last_error().decode())


def plan(L, N, R, tile=0, subsweeps=0, engine=ENGINE_AUTO, lanes=0, sm_count=0, cluster=0, poisson=False, multisurface=False):
    """rsos_plan: what rsos_init would choose for these arguments (host only, no device needed)."""
    o = RsosOpts(int(tile), int(subsweeps), 0, int(engine), None, None, 0, int(lanes), int(bool(poisson)), int(cluster), int(bool(multisurface)))
    a = (C.c_uint64 * 9)()
    _check(load().rsos_plan(int(L), int(N), int(R), C.byref(o), int(sm_count), a))
    return {"mode": "DT" if a[0] else "RS", "engine": ENGINE_NAMES[a[1]], "S": a[2], "K": a[3], "pass_tiles": a[4],
            "lanes": a[5], "packed_bits": a[6], "launches_per_mcs": a[7], "cluster": a[8]}


def philox(ctr, key):
    """Device Philox4x32-10 of n (counter, key) pairs: ctr (n,4) uint32, key (n,2) uint32 -> (n,4)."""
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    assert len(ctr) == len(key)
    out = np.empty_like(ctr)
    _check(load().rsos_philox(ctr.ctypes.data, key.ctypes.data, out.ctypes.data, len(ctr)))
    return out


def sums_static(d_heights, L, R, d_S1=None, d_S2=None, d_maxabs=None, stream=None):
    """rsos_sums_static: S1, S2 and max |h| of R surfaces that already sit in device memory, written to device arrays
    the caller owns, without any allocation by the library (see include/rsos.h: it exists for callers that cannot
    reach the CUDA allocator -- all device memory belongs to another pool -- or cannot afford its device-wide stall).

    Every pointer is a device address as a Python int (tensor.data_ptr()); the outputs hold R int64 / uint64 / uint32.
    R <= STATIC_MAX_R.  Asynchronous on `stream` (a cudaStream_t as int, None = the legacy default stream); all calls
    on a device share one fixed scratch array, so calls that could overlap on the GPU must be ordered by the caller.
    The first call on a device does a one-time address look-up; make it before any stream capture."""
    _check(load().rsos_sums_static(d_heights or None, int(L), int(R), d_S1 or None, d_S2 or None, d_maxabs or None, stream or None))


class Rsos:
    """rsos_init / rsos_advance / rsos_width ... with the same names as the C ABI.

    d_heights: optional device pointer (int) of an R*L*L int32 buffer, e.g. tensor.data_ptr();
    stream: optional cudaStream_t as int, e.g. torch.cuda.current_stream().cuda_stream.
    """

    def __init__(self, L, N, R, seed, tile=0, subsweeps=0, first_real=0, engine=ENGINE_AUTO,
                 d_heights=None, stream=None, device=None, lanes=0, cluster=0, poisson=False, multisurface=False):
        self._l = load()
        self.L, self.N, self.R, self.seed = int(L), int(N), int(R), int(seed)
        o = RsosOpts(int(tile), int(subsweeps), int(first_real), int(engine), d_heights or None,
                     stream or None, 0 if device is None else int(device) + 1, int(lanes), int(bool(poisson)), int(cluster), int(bool(multisurface)))
        self._c = C.c_void_p()
        _check(self._l.rsos_init(C.byref(self._c), self.L, self.N, self.R, self.seed, C.byref(o)))

    def close(self):
        if getattr(self, "_c", None):
            self._l.rsos_free(self._c)
            self._c = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def advance(self, mcs):
        _check(self._l.rsos_advance(self._c, int(mcs)))

    def sums(self):
        S1 = np.empty(self.R, dtype=np.int64)
        S2 = np.empty(self.R, dtype=np.uint64)
        acc = np.empty(self.R, dtype=np.int64)
        _check(self._l.rsos_sums(self._c, S1.ctypes.data, S2.ctypes.data, acc.ctypes.data))
        return S1, S2, acc

    def width(self):
        W2 = np.empty(self.R, dtype=np.float64)
        hm = np.empty(self.R, dtype=np.float64)
        _check(self._l.rsos_width(self._c, W2.ctypes.data, hm.ctypes.data))
        return W2, hm

    def moments(self):
        """(base[R] int64, M[R,4] python ints): M[r][k-1] = sum (h - base[r])^k, exact."""
        base = np.empty(self.R, dtype=np.int64)
        raw = np.empty((self.R, 4, 2), dtype=np.uint64)
        _check(self._l.rsos_moments(self._c, base.ctypes.data, raw.ctypes.data))
        M = []
        for r in range(self.R):
            row = []
            for k in range(4):
                v = int(raw[r, k, 0]) | (int(raw[r, k, 1]) << 64)
                row.append(v - (1 << 128) if v >> 127 else v)
            M.append(row)
        return base, M

    def height_moments(self):
        """(hbar[R], phi[R,3]): mean height and the central moments Phi^2, Phi^3, Phi^4 of every surface (Eq. 13)."""
        hbar = np.empty(self.R, dtype=np.float64)
        phi = np.empty((self.R, 3), dtype=np.float64)
        _check(self._l.rsos_height_moments(self._c, hbar.ctypes.data, phi.ctypes.data))
        return hbar, phi

    def heights(self, r0=0, nr=None, out=None):
        nr = self.R - r0 if nr is None else nr
        if out is None:
            out = np.empty((nr, self.L, self.L), dtype=np.int32)
        assert out.dtype == np.int32 and out.flags.c_contiguous and out.size == nr * self.L * self.L
        _check(self._l.rsos_get_heights(self._c, r0, nr, out.ctypes.data))
        return out

    def set_state(self, heights, t, accepted=None, r0=0):
        heights = np.ascontiguousarray(heights, dtype=np.int32).reshape(-1, self.L, self.L)
        acc = None if accepted is None else np.ascontiguousarray(accepted, dtype=np.int64)
        _check(self._l.rsos_set_state(self._c, r0, heights.shape[0], heights.ctypes.data, int(t),
                                      None if acc is None else acc.ctypes.data))

    @property
    def t(self):
        t = C.c_uint64()
        _check(self._l.rsos_time(self._c, C.byref(t)))
        return t.value

    def info(self):
        a = (C.c_uint64 * 12)()
        _check(self._l.rsos_info(self._c, a))
        return {"mode": "DT" if a[0] else "RS", "engine": ENGINE_NAMES[a[1]], "S": a[2], "K": a[3],
                "launches": a[4], "sm_count": a[5], "smem_bytes": a[6], "blocks": a[7], "lanes": a[8],
                "packed_bits": a[9], "cluster": a[10], "int32_allocated": bool(a[11])}

    def device_heights(self):
        d = C.c_void_p()
        _check(self._l.rsos_device_heights(self._c, C.byref(d)))
        return d.value

    def kernel_time(self, enable=True):
        """(ms_total, launches) of the rsos_advance calls since timing was enabled."""
        ms, n = C.c_double(), C.c_uint64()
        _check(self._l.rsos_kernel_time(self._c, int(bool(enable)), C.byref(ms), C.byref(n)))
        return ms.value, n.value
