"""GPU test of the no-allocation entry point `mpmc_contact_histogram_noalloc` (include/mpmc.h): the contact histogram
 with the kernels' scratch in a static device array inside the library instead of the workspace.
Checked against the existing path (`mpmc_pressure_contact`) on the same states: integer counts, so the bar is
bit-exact, as in the parity tests.  This file sorts last on purpose (the suite runs with `pytest -x`); it needs
nothing from the other test files and passes alone in a fresh process as well as after them."""
import numpy as np
import pytest

from paper_1211_1646_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_1211_1646_b200 import build
    build.build()
    return torch


def make(torch, name, fp32):
    from paper_1211_1646_b200.binding import Mpmc
    w = I.CONFIGS[name]
    xy, box = I.workload_inputs(w)
    g = Mpmc(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=fp32)
    g.load_positions(torch.as_tensor(xy, device="cuda"))
    return g


def as_u64(t):
    return t.cpu().numpy().view(np.uint64)


@pytest.mark.parametrize("fp32", [True, False])
def test_two_calls_in_a_row_match_the_existing_path(torch_cuda, fp32):
    g = make(torch_cuda, "C2", fp32)
    g.sweep(20)
    # first call: the paper's bins (L384: 200 bins of 1e-4 sigma ... here wider so that every bin is populated)
    want1 = g.contact_histogram(0.0005, 200)
    got1 = g.contact_histogram_noalloc(0.0005, 200)
    assert np.array_equal(as_u64(got1), want1) and want1.sum() > 1000
    # second call, straight after it: another state, FEWER and wider bins — the array still holds the first call's
    # 200 counts, so this fails unless the call clears what it uses
    g.sweep(7)
    want2 = g.contact_histogram(0.005, 20)
    got2 = g.contact_histogram_noalloc(0.005, 20)
    assert np.array_equal(as_u64(got2), want2) and want2.sum() > 1000
    assert not np.array_equal(want2, want1[:20])
    # and a third, with more bins than the second, into a caller-owned tensor that is larger than needed
    out = torch_cuda.full((300,), -1, dtype=torch_cuda.int64, device="cuda")
    g.contact_histogram_noalloc(0.001, 256, out=out)
    assert np.array_equal(as_u64(out[:256]), g.contact_histogram(0.001, 256))
    assert bool((out[256:] == -1).all())               # nothing written past nbins
    # the existing path is untouched by all this
    assert np.array_equal(g.contact_histogram(0.005, 20), want2)


def test_contexts_share_the_array_when_their_calls_do_not_overlap(torch_cuda):
    a = make(torch_cuda, "C1", False)
    b = make(torch_cuda, "C2", True)
    a.sweep(5); b.sweep(5)
    for _ in range(2):
        ha = a.contact_histogram_noalloc(0.01, 50)
        torch_cuda.cuda.synchronize()                  # two contexts = two streams: order the calls (they share the array)
        hb = b.contact_histogram_noalloc(0.002, 100)
        torch_cuda.cuda.synchronize()
        assert np.array_equal(as_u64(ha), a.contact_histogram(0.01, 50))
        assert np.array_equal(as_u64(hb), b.contact_histogram(0.002, 100))
        a.sweep(3); b.sweep(3)


def test_sizes_beyond_the_maximum_are_rejected(torch_cuda):
    from paper_1211_1646_b200 import binding
    g = make(torch_cuda, "C1", True)
    out = torch_cuda.full((binding.NOALLOC_MAX_BINS + 8,), -1, dtype=torch_cuda.int64, device="cuda")
    with pytest.raises(binding.MpmcError) as e:
        g.contact_histogram_noalloc(0.001, binding.NOALLOC_MAX_BINS + 1, out=out)
    assert e.value.code == binding.ERR_TOO_LARGE and "1024" in str(e.value)
    assert bool((out == -1).all())                     # nothing was launched
    full = g.contact_histogram_noalloc(0.0002, binding.NOALLOC_MAX_BINS, out=out)     # the maximum itself is fine
    assert np.array_equal(as_u64(full[:binding.NOALLOC_MAX_BINS]), g.contact_histogram(0.0002, binding.NOALLOC_MAX_BINS))
    with pytest.raises(binding.MpmcError) as e:        # bad arguments are still plain argument errors
        g.contact_histogram_noalloc(0.0, 10)
    assert e.value.code == -1
