"""ctypes loader for the CPU oracle (oracle/rsos_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It imports nothing from
paper_1605_02620_b200 and the CUDA path imports nothing from here.

All method arithmetic lives in the C file (each function there cites PAPER.md / SURVEY 8c.1);
this module only builds it with gcc and marshals numpy arrays.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rsos_oracle.c")
_LIB = os.path.join(_HERE, "librsos_oracle.so")
_lib = None


def build(force=False):
    """Compile the oracle with gcc -O2 -fopenmp (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        l = C.CDLL(build())
        u32, u64, i64, i32p = C.c_uint32, C.c_uint64, C.c_int64, C.POINTER(C.c_int32)
        vp = C.c_void_p
        l.rsos_oracle_philox.argtypes = [C.POINTER(u32), C.POINTER(u32), C.POINTER(u32)]
        l.rsos_oracle_philox.restype = None
        l.rsos_oracle_attempt.argtypes = [i32p, u32, i64, u32, u32]
        l.rsos_oracle_attempt.restype = C.c_int
        l.rsos_oracle_violations.argtypes = [i32p, u32, i64]
        l.rsos_oracle_violations.restype = i64
        l.rsos_oracle_create.argtypes = [u32, i64, u32, u64, u32, u32, u32]
        l.rsos_oracle_create.restype = vp
        l.rsos_oracle_free.argtypes = [vp]
        l.rsos_oracle_free.restype = None
        l.rsos_oracle_set_debug.argtypes = [vp, C.c_int, u64, C.c_int]
        l.rsos_oracle_set_debug.restype = None
        l.rsos_oracle_debug_violations.argtypes = [vp]
        l.rsos_oracle_debug_violations.restype = i64
        l.rsos_oracle_mode_dt.argtypes = [vp]
        l.rsos_oracle_mode_dt.restype = C.c_int
        l.rsos_oracle_advance.argtypes = [vp, u64]
        l.rsos_oracle_advance.restype = C.c_int
        l.rsos_oracle_threads.argtypes = [vp]
        l.rsos_oracle_threads.restype = C.c_int
        l.rsos_oracle_sums.argtypes = [vp, vp, vp, vp]
        l.rsos_oracle_sums.restype = C.c_int
        l.rsos_oracle_width.argtypes = [vp, vp, vp]
        l.rsos_oracle_width.restype = C.c_int
        l.rsos_oracle_get_heights.argtypes = [vp, u32, u32, vp]
        l.rsos_oracle_get_heights.restype = C.c_int
        l.rsos_oracle_set_state.argtypes = [vp, u32, u32, vp, u64, vp]
        l.rsos_oracle_set_state.restype = C.c_int
        l.rsos_oracle_time.argtypes = [vp]
        l.rsos_oracle_time.restype = u64
        l.rsos_oracle_last_error.restype = C.c_char_p
        l.rsos_oracle_height_moments.argtypes = [vp, u32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        l.rsos_oracle_height_moments.restype = C.c_int
        l.rsos_oracle_power_sums.argtypes = [vp, u32, i64, C.POINTER(u64)]
        l.rsos_oracle_power_sums.restype = C.c_int
        l.rsos_oracle_poisson4.argtypes = [u32]
        l.rsos_oracle_poisson4.restype = u32
        l.rsos_oracle_set_poisson.argtypes = [vp, C.c_int]
        l.rsos_oracle_set_poisson.restype = C.c_int
        l.rsos_oracle_set_multisurface.argtypes = [vp, C.c_int]
        l.rsos_oracle_set_multisurface.restype = C.c_int
        l.rsos_oracle_bounded.argtypes = [u32, u32, C.POINTER(C.c_int)]
        l.rsos_oracle_bounded.restype = u32
        l.rsos_oracle_bounded_census.argtypes = [u32, vp, C.POINTER(u64)]
        l.rsos_oracle_bounded_census.restype = None
        _lib = l
    return _lib


def poisson4(w):
    """Attempt count of the Poisson variant DTP for the 32-bit word w."""
    return int(lib().rsos_oracle_poisson4(int(w) & 0xFFFFFFFF))


def bounded(v, n):
    """One step of the exactly uniform bounded draw: (value in [0, n), accepted?)."""
    ok = C.c_int()
    r = lib().rsos_oracle_bounded(int(v) & 0xFFFFFFFF, int(n), C.byref(ok))
    return int(r), bool(ok.value)


def bounded_census(n):
    """(counts[n], rejected) of the bounded draw over all 2^32 words (a few seconds)."""
    counts = np.zeros(int(n), dtype=np.uint64)
    rej = C.c_uint64()
    lib().rsos_oracle_bounded_census(int(n), counts.ctypes.data, C.byref(rej))
    return counts, int(rej.value)


def philox(ctr, key):
    """Philox4x32-10 of one (counter, key); returns 4 uint32 as a numpy array."""
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().rsos_oracle_philox(c, k, o)
    return np.array(list(o), dtype=np.uint32)


def attempt(h, N, x, y):
    """One deposition attempt (Eq. 6) on the 2-D int32 array h (modified in place)."""
    assert h.dtype == np.int32 and h.flags.c_contiguous and h.ndim == 2 and h.shape[0] == h.shape[1]
    return lib().rsos_oracle_attempt(h.ctypes.data_as(C.POINTER(C.c_int32)), h.shape[0], int(N), int(x), int(y))


def violations(h, N):
    h = np.ascontiguousarray(h, dtype=np.int32)
    return lib().rsos_oracle_violations(h.ctypes.data_as(C.POINTER(C.c_int32)), h.shape[0], int(N))


class Oracle:
    """Same five logical operations as the C-ABI library (init / advance / width / sums / state)."""

    def __init__(self, L, N, R, seed, tile=64, subsweeps=1, first_real=0, threads=0,
                 check_each=False, shuffle_seed=0, poisson=False, multisurface=False):
        self.L, self.N, self.R, self.seed = int(L), int(N), int(R), int(seed)
        self._l = lib()
        self._c = self._l.rsos_oracle_create(self.L, self.N, self.R, self.seed, int(tile), int(subsweeps),
                                             int(first_real))
        if not self._c:
            raise ValueError("rsos_oracle_create: " + self._l.rsos_oracle_last_error().decode())
        self._l.rsos_oracle_set_debug(self._c, int(bool(check_each)), int(shuffle_seed), int(threads))
        if poisson and self._l.rsos_oracle_set_poisson(self._c, 1) != 0:
            raise ValueError("rsos_oracle_set_poisson: " + self._l.rsos_oracle_last_error().decode())
        if multisurface and self._l.rsos_oracle_set_multisurface(self._c, 1) != 0:
            raise ValueError("rsos_oracle_set_multisurface: " + self._l.rsos_oracle_last_error().decode())

    def close(self):
        if self._c:
            self._l.rsos_oracle_free(self._c)
            self._c = None

    __del__ = close

    @property
    def mode(self):
        return "DT" if self._l.rsos_oracle_mode_dt(self._c) else "RS"

    @property
    def threads(self):
        return self._l.rsos_oracle_threads(self._c)

    @property
    def t(self):
        return self._l.rsos_oracle_time(self._c)

    def advance(self, mcs):
        if self._l.rsos_oracle_advance(self._c, int(mcs)) != 0:
            raise ValueError("rsos_oracle_advance: " + self._l.rsos_oracle_last_error().decode())

    def sums(self):
        S1 = np.zeros(self.R, dtype=np.int64)
        S2 = np.zeros(self.R, dtype=np.uint64)
        acc = np.zeros(self.R, dtype=np.int64)
        self._l.rsos_oracle_sums(self._c, S1.ctypes.data, S2.ctypes.data, acc.ctypes.data)
        return S1, S2, acc

    def width(self):
        W2 = np.zeros(self.R, dtype=np.float64)
        hm = np.zeros(self.R, dtype=np.float64)
        self._l.rsos_oracle_width(self._c, W2.ctypes.data, hm.ctypes.data)
        return W2, hm

    def heights(self, r0=0, nr=None):
        nr = self.R - r0 if nr is None else nr
        out = np.empty((nr, self.L, self.L), dtype=np.int32)
        if self._l.rsos_oracle_get_heights(self._c, r0, nr, out.ctypes.data) != 0:
            raise ValueError("bad realization range")
        return out

    def set_state(self, heights, t, accepted=None, r0=0):
        heights = np.ascontiguousarray(heights, dtype=np.int32).reshape(-1, self.L, self.L)
        acc = None if accepted is None else np.ascontiguousarray(accepted, dtype=np.int64)
        if self._l.rsos_oracle_set_state(self._c, r0, heights.shape[0], heights.ctypes.data, int(t),
                                         None if acc is None else acc.ctypes.data) != 0:
            raise ValueError("bad realization range")

    def height_moments(self, r):
        """(hbar, [Phi^2, Phi^3, Phi^4]) of the heights of realization r: Eq. (13) by definition."""
        out = (C.c_double * 3)()
        hb = C.c_double()
        if self._l.rsos_oracle_height_moments(self._c, int(r), out, C.byref(hb)) != 0:
            raise ValueError("bad realization")
        return hb.value, [out[0], out[1], out[2]]

    def power_sums(self, r, base):
        """[M1..M4] with M_k = sum (h - base)^k as exact python ints."""
        out = (C.c_uint64 * 8)()
        if self._l.rsos_oracle_power_sums(self._c, int(r), int(base), out) != 0:
            raise ValueError("bad realization")
        res = []
        for k in range(4):
            v = int(out[2 * k]) | (int(out[2 * k + 1]) << 64)
            res.append(v - (1 << 128) if v >> 127 else v)
        return res

    def debug_violations(self):
        return self._l.rsos_oracle_debug_violations(self._c)
