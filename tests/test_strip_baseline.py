"""The OpenMP strip CPU baseline (oracle/strip_omp.cpp) against the single-threaded oracle: cells of a
checkerboard set are independent (L48) and the shift is double-buffered (L350), so the strips must reproduce the oracle's
trajectory bit for bit, whatever the number of threads."""
import numpy as np
import pytest

from paper_1211_1646_b200 import inputs as I


@pytest.mark.parametrize("fp32", [False, True])
@pytest.mark.parametrize("threads", [1, 3, 8])
def test_strips_reproduce_the_oracle(oracle_mod, fp32, threads):
    oracle_mod.build_strip()
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    o = oracle_mod.Oracle(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=fp32)
    s = oracle_mod.StripBaseline(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=fp32, threads=threads)
    assert s.threads == threads and (s.mx, s.my, s.wx, s.wy) == (o.mx, o.my, o.wx, o.wy)
    o.load_positions(xy); s.load_positions(xy)
    for k in (1, 7, 12):
        o.sweep(k); s.sweep(k)
        so, ss = o.debug_state(), s.debug_state()
        for key in ("counts", "slab", "ids", "accept_mask"):
            assert np.array_equal(so[key], ss[key]), key
        assert (so["origin"], so["sweep"], so["digest"]) == (ss["origin"], ss["sweep"], ss["digest"])
        assert o.acceptance() == s.acceptance()
    assert np.array_equal(o.get_positions(), s.get_positions())
    assert np.array_equal(o.contact_histogram(0.005, 20), s.contact_histogram(0.005, 20))


def test_strips_in_the_papers_regime(oracle_mod):
    # cells up to four disks, disc-shaped proposal, ablation flags: the options travel through the shared code
    xy, box = I.jittered_lattice(48, 0.698, seed=2)
    kw = dict(fp32=True, w_target=1.40, disc=True, particle_shuffle=False)
    o = oracle_mod.Oracle(48 * 48, box, 1.0, 0.16, 4, 3, **kw)
    s = oracle_mod.StripBaseline(48 * 48, box, 1.0, 0.16, 4, 3, threads=4, **kw)
    o.load_positions(xy); s.load_positions(xy)
    o.sweep(15); s.sweep(15)
    so, ss = o.debug_state(), s.debug_state()
    assert np.array_equal(so["slab"], ss["slab"]) and np.array_equal(so["ids"], ss["ids"]) and so["digest"] == ss["digest"]
    assert so["counts"].max() >= 3 and o.acceptance() == s.acceptance()
