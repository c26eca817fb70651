"""Thin Python binding of include/mpmc.h (ctypes).  Argument marshalling only: every step of the path runs in
the CUDA kernels behind the C ABI.  PyTorch supplies device memory and the stream, nothing else.

There is no CPU fallback: a missing library or a missing CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

FP64 = 0x1
FP32 = 0x2
DISC = 0x4
NO_PARTICLE_SHUFFLE = 0x8
NO_SET_SHUFFLE = 0x10
NO_RESIDENT = 0x20
DEBUG = 0x100
NOALLOC_MAX_BINS = 1024       # MPMC_NOALLOC_MAX_BINS of include/mpmc.h
ERR_TOO_LARGE = -8            # MPMC_ERR_TOO_LARGE

_u32, _u64, _dbl, _vp, _sz = C.c_uint32, C.c_uint64, C.c_double, C.c_void_p, C.c_size_t

# every symbol include/mpmc.h declares: name -> (restype, argtypes)
SYMBOLS = {
    "mpmc_workspace_bytes": (_sz, [_u64, C.POINTER(_dbl), _dbl, _u32]),
    "mpmc_workspace_bytes_ex": (_sz, [_u64, C.POINTER(_dbl), _dbl, _dbl, _u32]),
    "mpmc_create": (C.c_int, [C.POINTER(_vp), _u64, C.POINTER(_dbl), _dbl, _dbl, _u32, _u64, _u32, _vp, _sz, _vp]),
    "mpmc_create_ex": (C.c_int, [C.POINTER(_vp), _u64, C.POINTER(_dbl), _dbl, _dbl, _u32, _u64, _u32, _dbl, _vp, _sz, _vp]),
    "mpmc_destroy": (C.c_int, [_vp]),
    "mpmc_geometry": (C.c_int, [_vp, C.POINTER(_u32), C.POINTER(_dbl), C.POINTER(_dbl)]),
    "mpmc_load_positions": (C.c_int, [_vp, _vp]),
    "mpmc_sweep": (C.c_int, [_vp, _u64]),
    "mpmc_get_positions": (C.c_int, [_vp, _vp]),
    "mpmc_acceptance": (C.c_int, [_vp, C.POINTER(_u64)]),
    "mpmc_pressure_contact": (C.c_int, [_vp, _dbl, _u32, _u32, _vp, C.POINTER(_dbl), C.POINTER(_dbl)]),
    "mpmc_contact_histogram_noalloc": (C.c_int, [_vp, _dbl, _u32, _vp]),
    "mpmc_pressure_accumulate": (C.c_int, [_vp, _dbl, _u32]),
    "mpmc_pressure_accumulated": (C.c_int, [_vp, _u32, _vp, C.POINTER(_u64), C.POINTER(_dbl), C.POINTER(_dbl)]),
    "mpmc_pressure_reset": (C.c_int, [_vp]),
    "mpmc_pressure_from_histogram": (C.c_int, [_vp, _vp, _u64, _dbl, _u32, _u32, C.POINTER(_dbl), C.POINTER(_dbl)]),
    "mpmc_debug_sub_sweep": (C.c_int, [_vp, _u32]),
    "mpmc_debug_shift": (C.c_int, [_vp, _u32, _dbl]),
    "mpmc_debug_state": (C.c_int, [_vp, _vp, _vp, _vp, _vp, C.POINTER(_dbl), C.POINTER(_u64), C.POINTER(_u64)]),
    "mpmc_debug_path": (C.c_int, [_vp, C.POINTER(_u64)]),
    "mpmc_debug_config": (C.c_int, [_vp, C.POINTER(_u32)]),
    "mpmc_debug_phase_clocks": (C.c_int, [_vp, _vp, _u32, C.POINTER(_u32)]),
    "mpmc_debug_tiling": (C.c_int, [_u32, _u32, C.c_size_t, C.c_size_t, _u32, C.POINTER(_u32)]),
    "mpmc_debug_philox": (C.c_int, [_vp, C.POINTER(_u32), _vp, _u32, _vp]),
    "mpmc_strerror": (C.c_char_p, [C.c_int]),
    "mpmc_version": (C.c_char_p, []),
}

_lib = None


def library_path() -> str:
    return os.environ.get("MPMC_B200_LIB") or _build.LIB


def lib() -> C.CDLL:
    """Load libmpmc_b200.so (built in-tree by build.py / __graft_entry__.build()).  Raises if it is missing."""
    global _lib
    if _lib is None:
        path = library_path()
        if not os.path.exists(path):
            raise RuntimeError(f"{path} is missing: run `python -m paper_1211_1646_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(path)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


class MpmcError(RuntimeError):
    def __init__(self, code: int):
        super().__init__(f"mpmc error {code}: {lib().mpmc_strerror(code).decode()}")
        self.code = code


def _chk(code: int) -> None:
    if code != 0:
        raise MpmcError(code)


def workspace_bytes(N: int, box, sigma: float, fp32: bool, debug: bool = False, w_target: float = 0.0) -> int:
    b = (_dbl * 2)(float(box[0]), float(box[1]))
    flags = (FP32 if fp32 else FP64) | (DEBUG if debug else 0)
    return int(lib().mpmc_workspace_bytes_ex(int(N), b, float(sigma), float(w_target), flags))


class Mpmc:
    """mpmc_* calls on torch CUDA tensors.  Same call list as the C ABI."""

    def __init__(self, N: int, box, sigma: float, d: float, n_s: int, seed: int, fp32: bool = False,
                 debug: bool = False, w_target: float = 0.0, device="cuda:0", stream=None, disc: bool = False,
                 particle_shuffle: bool = True, set_shuffle: bool = True, resident: bool = True):
        """resident=False: MPMC_NO_RESIDENT (small systems on the tile / general kernels instead of the cluster-resident one)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1211_1646_b200 needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.N, self.fp32, self.debug, self.sigma = int(N), bool(fp32), bool(debug), float(sigma)
        self.flags = ((FP32 if fp32 else FP64) | (DEBUG if debug else 0) | (DISC if disc else 0)
                      | (0 if particle_shuffle else NO_PARTICLE_SHUFFLE) | (0 if set_shuffle else NO_SET_SHUFFLE)
                      | (0 if resident else NO_RESIDENT))
        nbytes = workspace_bytes(N, box, sigma, fp32, debug, w_target)
        if nbytes == 0:
            # let mpmc_create report the precise error code
            nbytes = 256
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            # The library's stream: a dedicated side stream by default (the legacy default stream cannot be
            # captured into a CUDA graph).  _enter/_exit order it against torch's current stream.
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
            self._h = _vp()
            b = (_dbl * 2)(float(box[0]), float(box[1]))
            _chk(lib().mpmc_create_ex(C.byref(self._h), self.N, b, float(sigma), float(d), int(n_s), int(seed),
                                      self.flags, float(w_target), self.workspace.data_ptr(), nbytes,
                                      self.stream.cuda_stream))
        m = (_u32 * 2)()
        w = (_dbl * 2)()
        Le = (_dbl * 2)()
        _chk(lib().mpmc_geometry(self._h, m, w, Le))
        self.mx, self.my = int(m[0]), int(m[1])
        self.wx, self.wy = float(w[0]), float(w[1])
        self.L_eff = (float(Le[0]), float(Le[1]))
        self.M = self.mx * self.my
        self.real = torch.float32 if fp32 else torch.float64

    def close(self) -> None:
        if getattr(self, "_h", None):
            lib().mpmc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _enter(self):
        cur = self.torch.cuda.current_stream(self.device)
        if cur != self.stream:
            self.stream.wait_stream(cur)

    def _exit(self):
        cur = self.torch.cuda.current_stream(self.device)
        if cur != self.stream:
            cur.wait_stream(self.stream)

    # --- the calls of include/mpmc.h -------------------------------------------------------------------
    def load_positions(self, xy) -> None:
        """xy: (N, 2) float64 CUDA tensor (device pointer passed through)."""
        t = self.torch
        assert xy.is_cuda and xy.dtype == t.float64 and tuple(xy.shape) == (self.N, 2) and xy.is_contiguous()
        with t.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_load_positions(self._h, xy.data_ptr()))
            self._exit()

    def sweep(self, k: int = 1) -> None:
        with self.torch.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_sweep(self._h, int(k)))
            self._exit()

    def get_positions(self, out=None):
        t = self.torch
        if out is None:
            out = t.empty((self.N, 2), dtype=t.float64, device=self.device)
        with t.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_get_positions(self._h, out.data_ptr()))
            self._exit()
        return out

    def acceptance(self):
        o = (_u64 * 4)()
        with self.torch.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_acceptance(self._h, o))
            self._exit()
        return tuple(int(v) for v in o)

    def pressure_contact(self, dr: float, nbins: int, degree: int):
        import numpy as np
        h = np.zeros(nbins, dtype=np.uint64)
        g0, ps = _dbl(), _dbl()
        with self.torch.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_pressure_contact(self._h, float(dr), int(nbins), int(degree), h.ctypes.data,
                                             C.byref(g0), C.byref(ps)))
            self._exit()
        return h, g0.value, ps.value

    def contact_histogram(self, dr: float, nbins: int):
        import numpy as np
        h = np.zeros(nbins, dtype=np.uint64)
        with self.torch.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_pressure_contact(self._h, float(dr), int(nbins), 0, h.ctypes.data, None, None))
            self._exit()
        return h

    def contact_histogram_noalloc(self, dr: float, nbins: int, out=None):
        """The pair histogram of mpmc_pressure_contact through the entry point that allocates nothing (its scratch is a
        static device array inside the library, at most NOALLOC_MAX_BINS bins; calls that overlap on the GPU race).
        out: int64 CUDA tensor of nbins elements owned by the caller (made here if None); asynchronous."""
        t = self.torch
        if out is None:
            out = t.empty(int(nbins), dtype=t.int64, device=self.device)
        assert out.is_cuda and out.dtype == t.int64 and out.is_contiguous() and out.numel() >= int(nbins)
        with t.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_contact_histogram_noalloc(self._h, float(dr), int(nbins), out.data_ptr()))
            self._exit()
        return out

    def pressure_accumulate(self, dr: float, nbins: int) -> None:
        """Add the current state's pair histogram to the device accumulator (asynchronous)."""
        with self.torch.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_pressure_accumulate(self._h, float(dr), int(nbins)))
            self._exit()

    def pressure_accumulated(self, degree: int, nbins: int, fit: bool = True):
        """(summed histogram, samples, g(sigma+), P*) of the accumulator; g and P* are None with fit=False."""
        import numpy as np
        h = np.zeros(nbins, dtype=np.uint64)
        n, g0, ps = _u64(), _dbl(), _dbl()
        with self.torch.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_pressure_accumulated(self._h, int(degree), h.ctypes.data, C.byref(n),
                                                 C.byref(g0) if fit else None, C.byref(ps) if fit else None))
            self._exit()
        return h, int(n.value), (g0.value if fit else None), (ps.value if fit else None)

    def pressure_reset(self) -> None:
        _chk(lib().mpmc_pressure_reset(self._h))

    def pressure_from_histogram(self, hist, samples: int, dr: float, degree: int):
        """(g(sigma+), P*) of eq. 4-6 on a histogram summed over `samples` configurations of this system (host arithmetic
        inside the library)."""
        import numpy as np
        h = np.ascontiguousarray(hist, dtype=np.uint64)
        g0, ps = _dbl(), _dbl()
        _chk(lib().mpmc_pressure_from_histogram(self._h, h.ctypes.data, int(samples), float(dr), len(h), int(degree),
                                                C.byref(g0), C.byref(ps)))
        return g0.value, ps.value

    # --- test hooks ------------------------------------------------------------------------------------
    def sub_sweep(self, checkerboard_set: int) -> None:
        with self.torch.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_debug_sub_sweep(self._h, int(checkerboard_set)))
            self._exit()

    def shift(self, direction: int, delta: float) -> None:
        with self.torch.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_debug_shift(self._h, int(direction), float(delta)))
            self._exit()

    def path_sweeps(self) -> tuple:
        """(sweeps done by the fused tile kernel, sweeps done by the general kernel) since the last load."""
        out = (_u64 * 2)()
        with self.torch.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_debug_path(self._h, out))
            self._exit()
        return int(out[0]), int(out[1])

    def config(self) -> dict:
        """How mpmc_sweep runs this context (mpmc_debug_config; host values only)."""
        out = (_u32 * 12)()
        _chk(lib().mpmc_debug_config(self._h, out))
        keys = ("tile_slots", "tiles", "ntx", "nty", "tile_threads", "tile_smem", "general_grid", "general_threads",
                "resident_ctas", "resident_cx", "resident_cy", "resident_smem")
        return dict(zip(keys, (int(v) for v in out)))

    def phase_clocks(self):
        """(tiles, marks) uint64 array of the tile kernel's clock marks in its last launch — for a context on the
        cluster-resident kernel (CTAs, 5): {sweeps, cycles in sub-sweeps, at barriers, in the shift, in the whole loop} of
        the last call; None unless the library was built with -DMPMC_PHASE_CLOCKS (mpmc_debug_phase_clocks)."""
        import numpy as np
        cfg = self.config()
        tiles = cfg["resident_ctas"] or cfg["tiles"]   # the cluster-resident kernel reports one row per CTA
        flat = np.zeros(max(tiles, 1) * 32, dtype=np.uint64)
        marks = _u32()
        with self.torch.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_debug_phase_clocks(self._h, flat.ctypes.data, tiles, C.byref(marks)))
            self._exit()
        if marks.value == 0:
            return None
        return flat[: tiles * marks.value].reshape(tiles, marks.value)

    def debug_state(self) -> dict:
        t = self.torch
        counts = t.empty(self.M, dtype=t.int32, device=self.device)
        slab = t.empty((self.M, 4, 2), dtype=self.real, device=self.device)
        ids = t.empty((self.M, 4), dtype=t.int32, device=self.device)
        mask = t.empty(self.M, dtype=t.int32, device=self.device) if self.debug else None
        origin = (_dbl * 2)()
        sw, dg = _u64(), _u64()
        with t.cuda.device(self.device):
            self._enter()
            _chk(lib().mpmc_debug_state(self._h, counts.data_ptr(), slab.data_ptr(), ids.data_ptr(),
                                        mask.data_ptr() if mask is not None else None, origin,
                                        C.byref(sw), C.byref(dg)))
            self._exit()
        import numpy as np
        return dict(counts=counts.cpu().numpy().view(np.uint32), slab=slab.cpu().numpy(),
                    ids=ids.cpu().numpy().view(np.uint32),
                    accept_mask=mask.cpu().numpy().view(np.uint32) if mask is not None else None,
                    origin=(origin[0], origin[1]), sweep=int(sw.value), digest=int(dg.value))


def tiling(hx: int, hy: int, cell_bytes: int = 16, smem_max: int = 226 * 1024, sms: int = 148):
    """(a, rows, plane stride, na, hyA, tiles) of the tiling the tile kernels would use (mpmc_debug_tiling); host
    arithmetic only.  None if the grid is too small to tile."""
    out = (_u32 * 6)()
    code = lib().mpmc_debug_tiling(int(hx), int(hy), int(cell_bytes), int(smem_max), int(sms), out)
    if code == -2:
        return None
    _chk(code)
    return tuple(int(v) for v in out)


def device_philox(ctr, key, device="cuda:0"):
    """Philox4x32-10 on the device (test hook).  ctr: (n, 4) integer array-like."""
    import numpy as np
    import torch
    c = torch.as_tensor(np.asarray(ctr, dtype=np.uint32).astype(np.int64), device=device).to(torch.int32).contiguous()
    n = c.shape[0]
    out = torch.empty((n, 4), dtype=torch.int32, device=device)
    k = (_u32 * 2)(int(key[0]) & 0xFFFFFFFF, int(key[1]) & 0xFFFFFFFF)
    with torch.cuda.device(device):
        _chk(lib().mpmc_debug_philox(c.data_ptr(), k, out.data_ptr(), n, torch.cuda.current_stream().cuda_stream))
    return out.cpu().numpy().view(np.uint32)
