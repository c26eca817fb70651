"""ORACLE — TEST INFRASTRUCTURE ONLY (ctypes front end of oracle_mpmc.cpp + the pressure fit).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from paper_1211_1646_b200 (the CUDA path) and the CUDA path imports
nothing from here.

The C++ file restates Algorithms 1, 2 and 4 of PAPER.md step by step; this file adds the host-side
pressure estimator of PAPER.md L366-382 (eq. 4-6) in numpy:
    g(R_i) = n[r_i] / (N rho 2 pi R_i dr)            (eq. 5; n[r_i] counts ORDERED pairs, so the
                                                      unordered histogram is doubled — reading A12)
    R_i    = (2/3) (r_{i+1}^3 - r_i^3) / (r_{i+1}^2 - r_i^2)          (eq. 6)
    fit g(R_i) by an unweighted least-squares polynomial of the given degree on (sigma, sigma + c],
    extrapolate to r = sigma (L382), and  P* = sigma^2 rho (1 + (pi/2) sigma^2 rho g(sigma+))  (eq. 4).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_mpmc.cpp")
_LIB = os.path.join(_HERE, "liboracle_mpmc.so")

FP64 = 1
FP32 = 2
NO_PARTICLE_SHUFFLE = 8     # ablations of PAPER.md section 2.4 / Table 1 (L114-142)
NO_SET_SHUFFLE = 16
LEAVE_CELL = 32   # ablation of PAPER.md section 2.4 pitfall 1 (L118-122): disks may leave their cell during a sub-sweep (oracle only)
DISC = 4      # trial displacement uniform in the disc of radius d instead of the square of reading A2

ERR = {0: "ok", -1: "bad argument", -2: "box too small", -4: "overlap or out-of-box input",
       -5: "cell overflow", -7: "no positions loaded"}


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (nothing contracted; the one FMA is written std::fma)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_STRIP_SRC = os.path.join(_HERE, "strip_omp.cpp")
_STRIP_LIB = os.path.join(_HERE, "liboracle_strip_omp.so")


def build_strip(force: bool = False) -> str:
    """The OpenMP strip baseline of PAPER.md L390 (strip_omp.cpp, which includes oracle_mpmc.cpp): g++ -O2 -fopenmp."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_STRIP_SRC))
    if force or not os.path.exists(_STRIP_LIB) or os.path.getmtime(_STRIP_LIB) < newest:
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
               "-o", _STRIP_LIB, _STRIP_SRC]
        subprocess.run(cmd, check=True)
    return _STRIP_LIB


_lib = None
_strip_lib = None


def _declare(L):
        u32, u64, dbl, vp = C.c_uint32, C.c_uint64, C.c_double, C.c_void_p
        L.oracle_create.argtypes = [C.POINTER(vp), u64, C.POINTER(dbl), dbl, dbl, u32, u64, u32, dbl]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_geometry.argtypes = [vp, C.POINTER(u32), C.POINTER(dbl), C.POINTER(dbl)]
        L.oracle_load_positions.argtypes = [vp, vp]
        L.oracle_sweep.argtypes = [vp, u64]
        L.oracle_get_positions.argtypes = [vp, vp]
        L.oracle_acceptance.argtypes = [vp, C.POINTER(u64)]
        L.oracle_contact_histogram.argtypes = [vp, dbl, u32, vp]
        L.oracle_debug_state.argtypes = [vp, vp, vp, vp, vp, C.POINTER(dbl), C.POINTER(u64), C.POINTER(u64)]
        L.oracle_sub_sweep.argtypes = [vp, u32]
        L.oracle_shift.argtypes = [vp, u32, dbl]
        L.oracle_philox4x32_10.argtypes = [C.POINTER(u32), C.POINTER(u32), C.POINTER(u32)]
        L.oracle_philox4x32_10.restype = None
        L.oracle_sweep_draws.argtypes = [u64, u64, C.POINTER(u32), C.POINTER(u32), C.POINTER(u32)]
        L.oracle_sweep_draws.restype = None
        L.oracle_visit_sequence.argtypes = [C.POINTER(u32), u32, u32, C.POINTER(u32)]
        L.oracle_visit_sequence.restype = None
        L.oracle_fisher_yates.argtypes = [C.POINTER(u32), u32, C.POINTER(u32)]
        L.oracle_fisher_yates.restype = None
        L.oracle_variate_sym_f32.argtypes = [u32]; L.oracle_variate_sym_f32.restype = C.c_float
        L.oracle_variate_sym_f64.argtypes = [u32]; L.oracle_variate_sym_f64.restype = C.c_double
        L.oracle_variate_unit_f32.argtypes = [u32]; L.oracle_variate_unit_f32.restype = C.c_float
        L.oracle_variate_unit_f64.argtypes = [u32]; L.oracle_variate_unit_f64.restype = C.c_double
        return L


def lib():
    global _lib
    if _lib is None:
        _lib = _declare(C.CDLL(build()))
    return _lib


def strip_lib():
    global _strip_lib
    if _strip_lib is None:
        L = _declare(C.CDLL(build_strip()))
        L.strip_create.argtypes = [C.POINTER(C.c_void_p), C.c_uint64, C.POINTER(C.c_double), C.c_double, C.c_double,
                                   C.c_uint32, C.c_uint64, C.c_uint32, C.c_double, C.c_int]
        L.strip_threads.restype = C.c_int
        _strip_lib = L
    return _strip_lib


class OracleError(RuntimeError):
    def __init__(self, code: int):
        super().__init__(f"oracle error {code}: {ERR.get(code, '?')}")
        self.code = code


def _chk(code: int) -> None:
    if code != 0:
        raise OracleError(code)


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def sweep_draws(seed: int, t: int):
    o = (C.c_uint32 * 4)()
    d = C.c_uint32()
    w = C.c_uint32()
    lib().oracle_sweep_draws(seed, t, o, C.byref(d), C.byref(w))
    return [int(v) for v in o], int(d.value), int(w.value)


def visit_sequence(perm, n_moves: int):
    p = (C.c_uint32 * len(perm))(*perm)
    o = (C.c_uint32 * n_moves)()
    lib().oracle_visit_sequence(p, len(perm), n_moves, o)
    return [int(v) for v in o]


def fisher_yates(a, words):
    arr = (C.c_uint32 * len(a))(*a)
    w = (C.c_uint32 * max(1, len(words)))(*words)
    lib().oracle_fisher_yates(arr, len(a), w)
    return [int(v) for v in arr]


class Oracle:
    """oracle_* calls with numpy host arrays.  Same call list as the product's `Mpmc` binding."""

    def __init__(self, N: int, box, sigma: float, d: float, n_s: int, seed: int, fp32: bool = False,
                 w_target: float = 0.0, disc: bool = False, particle_shuffle: bool = True, set_shuffle: bool = True,
                 leave_cell: bool = False):
        self._h = C.c_void_p()
        self.N = int(N)
        self.fp32 = bool(fp32)
        self.sigma = float(sigma)
        b = (C.c_double * 2)(float(box[0]), float(box[1]))
        flags = ((FP32 if fp32 else FP64) | (DISC if disc else 0) | (0 if particle_shuffle else NO_PARTICLE_SHUFFLE)
                 | (0 if set_shuffle else NO_SET_SHUFFLE) | (LEAVE_CELL if leave_cell else 0))
        self._create(b, sigma, d, n_s, seed, flags, float(w_target))
        m = (C.c_uint32 * 2)()
        w = (C.c_double * 2)()
        Le = (C.c_double * 2)()
        self._L.oracle_geometry(self._h, m, w, Le)
        self.mx, self.my = int(m[0]), int(m[1])
        self.wx, self.wy = float(w[0]), float(w[1])
        self.L_eff = (float(Le[0]), float(Le[1]))
        self.M = self.mx * self.my
        self.real = np.float32 if fp32 else np.float64

    def _create(self, b, sigma, d, n_s, seed, flags, w_target):
        self._L = lib()
        _chk(self._L.oracle_create(C.byref(self._h), self.N, b, sigma, d, n_s, seed, flags, w_target))

    def __del__(self):
        try:
            if self._h:
                self._L.oracle_destroy(self._h)
                self._h = None
        except Exception:
            pass

    def load_positions(self, xy: np.ndarray) -> None:
        xy = np.ascontiguousarray(xy, dtype=np.float64)
        assert xy.shape == (self.N, 2)
        _chk(self._L.oracle_load_positions(self._h, xy.ctypes.data))

    def sweep(self, k: int = 1) -> None:
        _chk(self._L.oracle_sweep(self._h, int(k)))

    def sub_sweep(self, checkerboard_set: int) -> None:
        _chk(self._L.oracle_sub_sweep(self._h, int(checkerboard_set)))

    def shift(self, direction: int, delta: float) -> None:
        _chk(self._L.oracle_shift(self._h, int(direction), float(delta)))

    def get_positions(self) -> np.ndarray:
        out = np.full((self.N, 2), np.nan, dtype=np.float64)
        _chk(self._L.oracle_get_positions(self._h, out.ctypes.data))
        return out

    def acceptance(self):
        o = (C.c_uint64 * 4)()
        _chk(self._L.oracle_acceptance(self._h, o))
        return tuple(int(v) for v in o)  # attempted, accepted, rej_boundary, rej_overlap

    def contact_histogram(self, dr: float, nbins: int) -> np.ndarray:
        h = np.zeros(nbins, dtype=np.uint64)
        _chk(self._L.oracle_contact_histogram(self._h, float(dr), int(nbins), h.ctypes.data))
        return h

    def pressure_contact(self, dr: float, nbins: int, degree: int):
        h = self.contact_histogram(dr, nbins)
        g0, p = pressure_from_histogram(h, self.N, self.L_eff, self.sigma, dr, degree)
        return h, g0, p

    def debug_state(self) -> dict:
        counts = np.zeros(self.M, dtype=np.uint32)
        slab = np.zeros((self.M, 4, 2), dtype=self.real)
        ids = np.zeros((self.M, 4), dtype=np.uint32)
        mask = np.zeros(self.M, dtype=np.uint32)
        origin = (C.c_double * 2)()
        t = C.c_uint64()
        dg = C.c_uint64()
        _chk(self._L.oracle_debug_state(self._h, counts.ctypes.data, slab.ctypes.data, ids.ctypes.data,
                                      mask.ctypes.data, origin, C.byref(t), C.byref(dg)))
        return dict(counts=counts, slab=slab, ids=ids, accept_mask=mask, origin=(origin[0], origin[1]),
                    sweep=int(t.value), digest=int(dg.value))


class StripBaseline(Oracle):
    """The OpenMP strip implementation of PAPER.md L390 (strip_omp.cpp): the oracle's Algorithms 2 and 4, one horizontal
    strip of cells per thread.  Same calls, same trajectory bit for bit; `threads` = OpenMP threads (0: all cores)."""

    def __init__(self, *args, threads: int = 0, **kw):
        self._threads = int(threads)
        super().__init__(*args, **kw)

    def _create(self, b, sigma, d, n_s, seed, flags, w_target):
        self._L = strip_lib()
        _chk(self._L.strip_create(C.byref(self._h), self.N, b, sigma, d, n_s, seed, flags, w_target, self._threads))
        self.threads = int(self._L.strip_threads())


def g_of_r(hist: np.ndarray, N: int, L_eff, sigma: float, dr: float):
    """eq. 5-6 of PAPER.md (L374-379); hist holds UNORDERED pair counts."""
    nb = len(hist)
    rho = N / (L_eff[0] * L_eff[1])
    r_lo = sigma + dr * np.arange(nb, dtype=np.float64)
    r_hi = sigma + dr * np.arange(1, nb + 1, dtype=np.float64)
    R = (2.0 / 3.0) * (r_hi ** 3 - r_lo ** 3) / (r_hi ** 2 - r_lo ** 2)
    g = 2.0 * hist.astype(np.float64) / (N * rho * 2.0 * np.pi * R * dr)
    return R, g, rho


def fit_contact(R: np.ndarray, g: np.ndarray, sigma: float, degree: int) -> float:
    """Unweighted least-squares polynomial in (R - sigma) of the given degree; value at R = sigma (L382)."""
    A = np.vander(R - sigma, degree + 1, increasing=True)
    coef, *_ = np.linalg.lstsq(A, g, rcond=None)
    return float(coef[0])


def pressure_from_histogram(hist, N, L_eff, sigma, dr, degree):
    R, g, rho = g_of_r(np.asarray(hist), N, L_eff, sigma, dr)
    g0 = fit_contact(R, g, sigma, degree)
    p_star = sigma ** 2 * rho * (1.0 + 0.5 * np.pi * sigma ** 2 * rho * g0)   # eq. 4 (L368)
    return g0, float(p_star)
