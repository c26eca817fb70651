"""ctypes front end of serial_mc.c (the independent serial-MC comparator; compiled on first use)."""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "serial_mc.c")
_LIB = os.path.join(_HERE, "libserial_mc.so")


def _lib():
    if not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"], check=True)
    L = C.CDLL(_LIB)
    L.serial_mc_pair_histograms.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_void_p,
                                            C.c_uint64, C.c_long, C.c_long, C.c_long, C.c_double, C.c_int,
                                            C.c_void_p, C.POINTER(C.c_double)]
    return L


def pair_histograms(xy0, L, sigma, d, seed, equil, nsamples, stride, rmax, nbins):
    xy0 = np.ascontiguousarray(xy0, dtype=np.float64)
    out = np.zeros((nsamples, nbins), dtype=np.float64)
    acc = C.c_double()
    rc = _lib().serial_mc_pair_histograms(len(xy0), L[0], L[1], sigma, d, xy0.ctypes.data, seed, equil, nsamples,
                                          stride, rmax, nbins, out.ctypes.data, C.byref(acc))
    assert rc == 0
    return out, acc.value
