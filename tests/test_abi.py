"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol that
include/mpmc.h declares, does its pure-host arithmetic, and fails loudly (no CPU fallback) without a GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1211_1646_b200 import build, binding
    build.build()
    return binding.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "mpmc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mpmc_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_all_exported(lib):
    from paper_1211_1646_b200 import binding
    names = declared_symbols()
    assert len(names) >= 17
    for n in names:
        assert hasattr(lib, n), n
        assert n in binding.SYMBOLS, f"{n} missing from the Python binding"
    assert sorted(binding.SYMBOLS) == names


def test_version_and_strerror(lib):
    assert b"sm_100a" in lib.mpmc_version()
    for code in range(0, -9, -1):
        assert lib.mpmc_strerror(code) and lib.mpmc_strerror(code) != b"unknown error"
    assert b"1024" in lib.mpmc_strerror(-8)          # MPMC_ERR_TOO_LARGE names the limit of the no-allocation entry point
    assert lib.mpmc_strerror(-99) == b"unknown error"


def test_workspace_bytes_host_arithmetic(lib):
    from paper_1211_1646_b200 import binding, inputs
    w = inputs.CONFIGS["C3"]
    box = inputs.box_for(w.n_side, w.phi)
    nb = binding.workspace_bytes(w.N, box, 1.0, fp32=True)
    Mq = (1152 // 2) * (998 // 2)
    # two buffers of 4 colours x 4 slot planes of float2 + ids + counts
    assert nb >= 2 * 16 * Mq * (8 + 4) + 2 * 4 * Mq
    assert nb < 1.1 * (2 * 16 * Mq * 12 + 2 * 4 * Mq + 4 * 4 * Mq) + (1 << 20)
    assert binding.workspace_bytes(w.N, box, 1.0, fp32=False) > nb
    assert binding.workspace_bytes(w.N, box, 1.0, fp32=True, debug=True) >= nb + 4 * 1152 * 998
    assert binding.workspace_bytes(w.N, (1.5, 10.0), 1.0, fp32=True) == 0      # box too small
    assert binding.workspace_bytes(0, box, 1.0, fp32=True) == 0
    b = (C.c_double * 2)(*box)
    assert lib.mpmc_workspace_bytes(w.N, b, 1.0, binding.FP32 | binding.FP64) == 0   # both precision bits
    # a wider target cell means fewer cells and a smaller workspace
    assert binding.workspace_bytes(w.N, box, 1.0, fp32=True, w_target=1.4) < nb


def test_argument_errors_without_gpu(lib):
    from paper_1211_1646_b200 import binding
    h = C.c_void_p()
    b = (C.c_double * 2)(10.0, 10.0)
    fake = C.c_void_p(0x10000)   # never dereferenced: argument checks come first
    assert lib.mpmc_create(C.byref(h), 0, b, 1.0, 0.1, 4, 1, binding.FP32, fake, 1 << 30, None) == -1
    assert lib.mpmc_create(C.byref(h), 10, b, 1.0, 0.1, 33, 1, binding.FP32, fake, 1 << 30, None) == -1
    assert lib.mpmc_create(C.byref(h), 10, b, 1.0, 0.1, 4, 1, 0, fake, 1 << 30, None) == -1
    small = (C.c_double * 2)(1.9, 10.0)
    assert lib.mpmc_create(C.byref(h), 10, small, 1.0, 0.1, 4, 1, binding.FP32, fake, 1 << 30, None) == -2
    assert lib.mpmc_create(C.byref(h), 10, b, 1.0, 0.1, 4, 1, binding.FP32, None, 1 << 30, None) == -3
    assert lib.mpmc_create(C.byref(h), 10, b, 1.0, 0.1, 4, 1, binding.FP32, fake, 16, None) == -3
    assert lib.mpmc_create(C.byref(h), 10, b, 1.0, 0.1, 4, 1, binding.FP32, C.c_void_p(0x10001), 1 << 30, None) == -3
    assert lib.mpmc_sweep(None, 1) == -1
    assert lib.mpmc_contact_histogram_noalloc(None, 0.1, 10, fake) == -1
    assert lib.mpmc_destroy(None) == 0


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1211_1646_b200 import binding
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.Mpmc(16, (10.0, 10.0), 1.0, 0.1, 4, 1)
    # and the C library itself reports MPMC_ERR_CUDA rather than computing anything
    h = C.c_void_p()
    b = (C.c_double * 2)(10.0, 10.0)
    assert binding.lib().mpmc_create(C.byref(h), 10, b, 1.0, 0.1, 4, 1, binding.FP32, C.c_void_p(0x10000), 1 << 30,
                                     None) == -6


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1211_1646_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert "oracle_mpmc" not in src and "liboracle" not in src, f
    orc = open(os.path.join(ROOT, "oracle", "oracle.py")).read() + open(os.path.join(ROOT, "oracle", "oracle_mpmc.cpp")).read()
    assert "paper_1211_1646_b200" not in orc.replace("paper_1211_1646_b200/csrc (the CUDA", "").replace(
        "imports nothing from paper_1211_1646_b200", "")
    assert "mpmc.h" not in orc


def test_tiling_of_the_tile_kernels_host_logic():
    """choose_tiling (csrc/mpmc.cu) through the mpmc_debug_tiling hook, no device: the tiles cover the grid exactly, every
    tile plus its halo of 5 fits the shared memory and is no wider than the grid (a loaded region must not overlap itself),
    and the busiest SM's work (waves x largest region) is not worse than a few obvious uniform alternatives."""
    import math
    from paper_1211_1646_b200 import binding as B
    smem, sms = 226 * 1024, 148
    for hx, hy, cb in [(576, 499, 16), (145, 126, 16), (43, 37, 32), (2298, 1990, 16), (618, 534, 32), (9, 7, 16), (6, 6, 16),
                       (1000, 8, 16), (8, 1000, 64), (576, 499, 18), (890, 770, 18)]:
        t = B.tiling(hx, hy, cb, smem, sms)
        assert t is not None, (hx, hy)
        a, rows, PS, na, hyA, tiles = t
        nb = rows - na
        assert 1 <= a <= hx and 1 <= na <= rows <= hy and tiles == na * a + nb * (a + 1)
        assert (nb == 0 and hyA == hy) or (0 < hyA < hy and tiles <= sms)          # mixed tilings only within one wave
        # the tiles as the kernel derives them (tile_box): rows of group A then of group B, each row split along x
        cells, worst, ps_max = 0, 0, 0
        groups = [(na, a, 0, hyA)] + ([(nb, a + 1, hyA, hy)] if nb else [])
        for nrow, ntx, h_lo, h_hi in groups:
            for r in range(nrow):
                h0, h1 = h_lo + (h_hi - h_lo) * r // nrow, h_lo + (h_hi - h_lo) * (r + 1) // nrow
                for tx in range(ntx):
                    TX, TY = 2 * (hx * (tx + 1) // ntx - hx * tx // ntx), 2 * (h1 - h0)
                    assert TX >= 2 and TY >= 2 and TX + 10 <= 2 * hx and TY + 10 <= 2 * hy
                    cells += TX * TY
                    worst = max(worst, (TX + 10) * (TY + 10))
                    ps_max = max(ps_max, ((TX + 10) // 2) * ((TY + 10) // 2))
        assert cells == 4 * hx * hy                                          # an exact cover
        assert ps_max <= PS and 4 * PS * cb <= smem                          # four colour planes of the largest tile fit
        cost = math.ceil(tiles / sms) * worst
        for ax, ay in [(1, 1), (a + 1, rows), (a, rows + 1), (max(1, a - 1), rows), (a, max(1, rows - 1)), (12, 12), (sms, 1)]:
            if ax > hx or ay > hy:
                continue
            ux, uy = 2 * math.ceil(hx / ax), 2 * math.ceil(hy / ay)
            if ux + 10 > 2 * hx or uy + 10 > 2 * hy or 4 * ((ux + 10) // 2) * ((uy + 10) // 2) * cb > smem:
                continue
            assert cost <= math.ceil(ax * ay / sms) * (ux + 10) * (uy + 10) * (1 + 1e-9), (hx, hy, t, ax, ay)
    a, rows, PS, na, hyA, tiles = B.tiling(576, 499, 18, smem, sms)          # the headline grid: all 148 SMs get a tile
    assert tiles == 148 and na < rows
    assert B.tiling(5, 40, 16, smem, sms) is None and B.tiling(40, 4, 16, smem, sms) is None   # under 12 cells across
    assert B.tiling(100, 100, 16, 4 * 36 * 16 - 1, sms) is None                                # not even a 2 x 2 tile fits
