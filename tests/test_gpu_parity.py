"""GPU parity tests (`-m gpu`): the CUDA path, called through the C ABI, against the CPU oracle on the same
seeded inputs.  Bar (BASELINE.json north_star): accept/reject sequences, counters, cell membership, slot order
and ids bit-exact; local coordinates bit-exact in both precisions (stronger than the stated |dx| <= 1e-12 /
1e-5 on unpacked positions, which is checked as well); every configuration overlap-free."""
import math

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


def make_pair(oracle_mod, torch, N, box, sigma, d, n_s, seed, fp32, xy, debug=True, w_target=0.0, disc=False,
              resident=False, **ablate):
    """resident=False keeps small systems on the tile / general kernels (MPMC_NO_RESIDENT), which is what most tests here
    are about; the cluster-resident kernel has its own tests below (test_resident_*)."""
    from paper_1211_1646_b200.binding import Mpmc
    o = oracle_mod.Oracle(N, box, sigma, d, n_s, seed, fp32=fp32, w_target=w_target, disc=disc, **ablate)
    g = Mpmc(N, box, sigma, d, n_s, seed, fp32=fp32, debug=debug, w_target=w_target, disc=disc, resident=resident, **ablate)
    assert (g.mx, g.my) == (o.mx, o.my) and (g.wx, g.wy) == (o.wx, o.wy) and g.L_eff == o.L_eff
    o.load_positions(xy)
    g.load_positions(torch.as_tensor(xy, device="cuda"))
    return o, g


def assert_same_state(o, g, fp32, check_mask=True, pos_tol=None):
    so, sg = o.debug_state(), g.debug_state()
    assert sg["sweep"] == so["sweep"]
    assert np.array_equal(sg["counts"], so["counts"])
    assert np.array_equal(sg["ids"], so["ids"])
    assert np.array_equal(sg["slab"].view(np.uint32 if fp32 else np.uint64),
                          so["slab"].view(np.uint32 if fp32 else np.uint64))      # bit-exact locals
    assert sg["origin"] == so["origin"]
    if check_mask and sg["accept_mask"] is not None:
        assert np.array_equal(sg["accept_mask"], so["accept_mask"])
        assert sg["digest"] == so["digest"]
    assert g.acceptance() == o.acceptance()
    po, pg = o.get_positions(), g.get_positions().cpu().numpy()
    tol = pos_tol if pos_tol is not None else (1e-5 if fp32 else 1e-12)
    assert np.abs(pg - po).max() <= tol
    assert np.array_equal(pg, po)      # same formula, same operands: in fact identical
    return so


def test_device_philox_matches_known_answers_and_oracle(oracle_mod, torch_cuda):
    from paper_1211_1646_b200.binding import device_philox
    kat = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344]]
    keys = [(0, 0), (0xFFFFFFFF, 0xFFFFFFFF), (0xa4093822, 0x299f31d0)]
    want = [[0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8], [0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd],
            [0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1]]
    for c, k, w in zip(kat, keys, want):
        assert device_philox([c], k)[0].tolist() == w
    rng = np.random.default_rng(5)
    ctr = rng.integers(0, 2 ** 32, size=(1000, 4), dtype=np.uint64)
    got = device_philox(ctr, (123, 456))
    for i in range(0, 1000, 37):
        assert got[i].tolist() == oracle_mod.philox4x32_10(ctr[i].tolist(), (123, 456))


@pytest.mark.parametrize("fp32", [False, True])
def test_pieces_load_subsweeps_shift(oracle_mod, torch_cuda, fp32):
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    o, g = make_pair(oracle_mod, torch_cuda, w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32, xy)
    assert_same_state(o, g, fp32)                      # cell-list build
    for q in (2, 0, 3, 1):                             # one sub-sweep per checkerboard set
        o.sub_sweep(q); g.sub_sweep(q)
        assert_same_state(o, g, fp32)
    for direction in range(4):                         # the four shift directions
        delta = 0.31 * (o.wx if direction < 2 else o.wy)
        o.shift(direction, delta); g.shift(direction, delta)
        assert_same_state(o, g, fp32)
    o.shift(0, 0.0); g.shift(0, 0.0)                   # delta = 0 is allowed (reading A5)
    assert_same_state(o, g, fp32)


@pytest.mark.parametrize("workload", ["C1", "C3s"])
def test_sweeps_after_test_hook_shifts(oracle_mod, torch_cuda, workload):
    """The host tells every tile-kernel launch which buffer holds its sweep's state; a shift made through the test hook
    flips the buffer at an unchanged sweep index, an odd number of sweeps flips it too.  C3s: a system large enough for
    the sorted variant, which starts from that hint before it has seen the control block."""
    if workload == "C1":
        w = I.CONFIGS["C1"]
        N, sigma, d, n_s, seed, fp32 = w.N, w.sigma, w.d, w.n_s, w.seed, w.fp32
        xy, box = I.workload_inputs(w)
    else:
        n = 704                                        # ~3 700 cells per tile region: the sorted variant
        N, sigma, d, n_s, seed, fp32 = n * n, 1.0, 0.08, 4, 11, True
        xy, box = I.jittered_lattice(n, 0.716, sigma, seed=seed)
    o, g = make_pair(oracle_mod, torch_cuda, N, box, sigma, d, n_s, seed, fp32, xy)
    done = 0
    for k, direction in ((3, 1), (2, 2), (1, 0), (4, 3)):
        o.sweep(k); g.sweep(k); done += k
        assert_same_state(o, g, fp32)
        delta = 0.27 * (o.wx if direction < 2 else o.wy)
        o.shift(direction, delta); g.shift(direction, delta)
        assert_same_state(o, g, fp32)
    o.sweep(5); g.sweep(5); done += 5
    assert_same_state(o, g, fp32)
    assert g.path_sweeps() == (done, 0)                # every sweep on the fused tile kernel, none refused
    if workload == "C3s":
        assert g.config()["tile_slots"] == 2


@pytest.mark.parametrize("fp32", [False, True])
def test_c1_100_sweeps_bit_exact(oracle_mod, torch_cuda, fp32):
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    o, g = make_pair(oracle_mod, torch_cuda, w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32, xy)
    for k in (1, 1, 3, 16, 17, 62):                    # several call sizes: one tile-kernel launch per sweep
        o.sweep(k); g.sweep(k)
        st = assert_same_state(o, g, fp32)
    assert st["sweep"] == 100
    assert g.path_sweeps() == (100, 0)                 # every sweep on the fused tile kernel
    att, acc, rb, ro = g.acceptance()
    assert att == acc + rb + ro and acc > 0 and rb > 0 and ro > 0


# ---- the cluster-resident kernel for small systems (cluster.cuh): all sweeps of a call in one launch of one cluster ----
@pytest.mark.parametrize("fp32", [False, True])
def test_resident_c1_100_sweeps_bit_exact(oracle_mod, torch_cuda, fp32):
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    o, g = make_pair(oracle_mod, torch_cuda, w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32, xy, resident=True)
    cfg = g.config()
    assert cfg["resident_ctas"] == cfg["resident_cx"] * cfg["resident_cy"] >= 1
    for k in (1, 1, 3, 16, 17, 62):                    # several call sizes: one launch per call
        o.sweep(k); g.sweep(k)
        st = assert_same_state(o, g, fp32)
    assert st["sweep"] == 100 and g.path_sweeps() == (100, 0)
    # pieces through the test hooks (general kernel on the global state) between resident calls
    o.sub_sweep(2); g.sub_sweep(2)
    o.shift(1, 0.3 * o.wx); g.shift(1, 0.3 * o.wx)
    o.sweep(5); g.sweep(5)
    assert_same_state(o, g, fp32)
    ho, _, _ = o.pressure_contact(0.005, 20, 2)
    assert np.array_equal(ho, g.contact_histogram(0.005, 20))


@pytest.mark.parametrize("n,phi,w_target,disc,fp32", [(26, 0.6, 0.0, False, True), (50, 0.716, 0.0, False, False),
                                                      (34, 0.3, 0.0, False, True), (64, 0.698, 1.4, True, True),
                                                      (46, 0.698, 1.4, False, False), (90, 0.716, 0.0, False, True),
                                                      (120, 0.65, 1.4, True, True)])
def test_resident_uneven_tiles_widths_and_proposals(oracle_mod, torch_cuda, n, phi, w_target, disc, fp32):
    """Grids that do not divide evenly among the cluster's CTAs, both cell regimes (cells of up to 4 disks), both
    proposals, dilute and dense."""
    xy, box = I.jittered_lattice(n, phi, 1.0, seed=3)
    o, g = make_pair(oracle_mod, torch_cuda, n * n, box, 1.0, 0.12, 4, 77, fp32, xy, w_target=w_target, disc=disc, resident=True)
    assert g.config()["resident_ctas"] >= 1
    for k in (1, 2, 9):
        o.sweep(k); g.sweep(k)
        assert_same_state(o, g, fp32)
    assert g.path_sweeps() == (12, 0)


@pytest.mark.parametrize("fp32", [False, True])
def test_resident_cells_with_three_disks_at_unit_width(oracle_mod, torch_cuda, fp32):
    # w ~ 1.13 sigma keeps the fast cell update (w < 1.15 sigma) while cells with THREE disks do occur: next to such a cell
    # the update takes the general routine, the shift the eight-candidate one (the recipe of
    # test_three_per_cell_with_two_register_slots, on the resident kernel)
    xy, box = I.jittered_lattice(64, 0.50, seed=6)
    o, g = make_pair(oracle_mod, torch_cuda, 4096, box, 1.0, 0.3, 4, 8, fp32, xy, w_target=1.12, resident=True)
    assert g.config()["resident_ctas"] >= 1 and g.config()["tile_slots"] == 2
    seen3 = False
    for _ in range(10):
        o.sweep(20); g.sweep(20)
        st = assert_same_state(o, g, fp32)
        seen3 |= st["counts"].max() >= 3
    assert seen3 and g.path_sweeps() == (200, 0)


@pytest.mark.parametrize("N,box,xy", [
    (1, (2.6, 2.6), [[0.3, 0.4]]),
    (2, (2.6, 2.9), [[0.5, 0.5], [1.8, 1.9]]),                 # mx = my = 2: neighbour at two image offsets
    (3, (4.3, 4.5), [[0.5, 0.5], [2.0, 2.0], [3.5, 0.9]]),
    (5, (9.7, 2.4), [[0.5, 0.5], [2.0, 1.9], [3.5, 0.9], [6.1, 1.2], [8.3, 0.4]]),     # 8 x 2 cells: tiles one cell high
])
@pytest.mark.parametrize("fp32", [False, True])
def test_resident_tiny_systems(oracle_mod, torch_cuda, N, box, xy, fp32):
    xy = np.array(xy, dtype=np.float64)
    o, g = make_pair(oracle_mod, torch_cuda, N, box, 1.0, 0.4, 4, 9, fp32, xy, resident=True)
    assert g.config()["resident_ctas"] >= 1
    for _ in range(5):
        o.sweep(40); g.sweep(40)
        assert_same_state(o, g, fp32)


@pytest.mark.parametrize("pshuf,sshuf", [(False, True), (True, False), (False, False)])
@pytest.mark.parametrize("w_target", [0.0, 1.40])
def test_resident_ablation_switches(oracle_mod, torch_cuda, pshuf, sshuf, w_target):
    xy, box = I.jittered_lattice(64, 0.66, seed=12)
    o, g = make_pair(oracle_mod, torch_cuda, 4096, box, 1.0, 0.2, 4, 3, True, xy, w_target=w_target,
                     particle_shuffle=pshuf, set_shuffle=sshuf, resident=True)
    assert g.config()["resident_ctas"] >= 1
    o.sweep(12); g.sweep(12)
    assert_same_state(o, g, True)


@pytest.mark.parametrize("name,fp32", [("S64", True), ("C1", False), ("P64", True)])
def test_resident_long_runs_in_one_launch(oracle_mod, torch_cuda, name, fp32):
    """2 000 sweeps in ONE launch (10 000 barriers between CTAs that read each other's shared memory): any ordering slip of
    the kernel's barrier (a CTA-scope fence and a relaxed arrive, cluster.cuh cl_sync) would change the trajectory."""
    w = I.CONFIGS[name]
    xy, box = I.workload_inputs(w)
    o, g = make_pair(oracle_mod, torch_cuda, w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32, xy, debug=False, w_target=w.w_target,
                     disc=w.disc, resident=True)
    assert g.config()["resident_ctas"] == 16
    for k in (2000, 1):
        o.sweep(k); g.sweep(k)
        assert_same_state(o, g, fp32)
    assert g.path_sweeps() == (2001, 0)


def test_resident_is_not_used_beyond_its_capacity_or_when_switched_off(oracle_mod, torch_cuda):
    from paper_1211_1646_b200.binding import Mpmc
    w = I.CONFIGS["C2"]                                # 73 080 cells: too many for one cluster
    xy, box = I.workload_inputs(w)
    assert Mpmc(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=True).config()["resident_ctas"] == 0
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    assert Mpmc(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=True, resident=False).config()["resident_ctas"] == 0
    assert Mpmc(w.N, box, w.sigma, w.d, 8, w.seed, fp32=True).config()["resident_ctas"] == 0      # n_s = 4 only
    assert Mpmc(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=True).config()["resident_ctas"] >= 1


@pytest.mark.parametrize("fp32", [False, True])
def test_c2_dense_fluid(oracle_mod, torch_cuda, fp32):
    w = I.CONFIGS["C2"]
    xy, box = I.workload_inputs(w)
    o, g = make_pair(oracle_mod, torch_cuda, w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32, xy)
    assert (g.mx, g.my) == (290, 252)
    o.sweep(40); g.sweep(40)
    assert_same_state(o, g, fp32)
    # contact pressure every 10 sweeps: histogram bit-exact, fit to rounding (config C2: bin width 0.005 sigma)
    for _ in range(2):
        o.sweep(10); g.sweep(10)
        ho, g0o, pso = o.pressure_contact(0.005, 20, 2)
        hg, g0g, psg = g.pressure_contact(0.005, 20, 2)
        assert np.array_equal(ho, hg) and ho.sum() > 1000
        assert g0g == pytest.approx(g0o, rel=1e-9) and psg == pytest.approx(pso, rel=1e-9)
    hg = g.contact_histogram(1e-4, 200)                # the paper's estimator parameters (L382)
    assert np.array_equal(hg, o.contact_histogram(1e-4, 200))


@pytest.mark.parametrize("fp32", [False, True])
@pytest.mark.parametrize("w_target", [0.0, 1.12, 1.40])
def test_contact_histogram_ranges(oracle_mod, torch_cuda, fp32, w_target):
    """a4 on its own: neighbourhood radius 1 and 2 (tiles in shared memory) and 3, 4 (general kernel), cells with 0..4
    disks, bins from the paper's 1e-4 sigma (L382) to coarse ones; counts identical to the oracle's."""
    xy, box = I.jittered_lattice(64, 0.55, seed=21)
    o, g = make_pair(oracle_mod, torch_cuda, 4096, box, 1.0, 0.3, 4, 6, fp32, xy, w_target=w_target)
    o.sweep(30); g.sweep(30)
    st = assert_same_state(o, g, fp32)
    if w_target > 1.0:
        assert st["counts"].max() >= 3
    for dr, nbins in [(0.005, 20), (1e-4, 200), (0.0004, 1000), (0.01, 250), (0.001, 4096), (0.6, 3)]:
        ho, hg = o.contact_histogram(dr, nbins), g.contact_histogram(dr, nbins)
        assert np.array_equal(ho, hg), (dr, nbins, int(ho.sum()), int(hg.sum()))
        assert ho.sum() > 0


@pytest.mark.parametrize("N,box,xy", [
    (2, (2.6, 2.9), [[0.5, 0.5], [1.8, 1.9]]),                 # mx = my = 2: every cell is met at several image offsets
    (3, (4.3, 4.5), [[0.5, 0.5], [2.0, 2.0], [3.5, 0.9]]),
    (5, (6.4, 3.3), [[0.4, 0.4], [1.6, 0.5], [2.9, 0.6], [4.3, 2.2], [5.5, 1.0]]),
])
@pytest.mark.parametrize("fp32", [False, True])
def test_contact_histogram_of_tiny_boxes(oracle_mod, torch_cuda, N, box, xy, fp32):
    xy = np.array(xy, dtype=np.float64)
    o, g = make_pair(oracle_mod, torch_cuda, N, box, 1.0, 0.4, 4, 9, fp32, xy)
    for _ in range(3):
        o.sweep(7); g.sweep(7)
        for dr, nbins in [(0.005, 20), (0.05, 20), (0.1, 25), (0.25, 20)]:    # radius 2, 2, 3-4, 5-6 cells: images of images
            assert np.array_equal(o.contact_histogram(dr, nbins), g.contact_histogram(dr, nbins)), (dr, nbins)


@pytest.mark.parametrize("fp32", [False, True])
def test_sample_averaged_pressure_estimator(oracle_mod, torch_cuda, fp32):
    """The paper's procedure (L384, eq. 5): histograms of many configurations are averaged, then fitted.  The accumulator
    and the fit live behind the C ABI; the oracle's estimator on the summed oracle histograms is the reference."""
    from paper_1211_1646_b200.binding import MpmcError
    xy, box = I.jittered_lattice(64, 0.66, seed=5)
    o, g = make_pair(oracle_mod, torch_cuda, 4096, box, 1.0, 0.15, 4, 2, fp32, xy)
    dr, nbins, degree = 1e-3, 40, 3
    with pytest.raises(MpmcError) as e:
        g.pressure_accumulated(degree, nbins)            # no sample yet
    assert e.value.code == -7
    total = np.zeros(nbins, dtype=np.uint64)
    for s in range(6):
        o.sweep(5); g.sweep(5)
        g.pressure_accumulate(dr, nbins)
        total += o.contact_histogram(dr, nbins)
    with pytest.raises(MpmcError) as e:
        g.pressure_accumulate(2 * dr, nbins)             # the bins are fixed by the first sample
    assert e.value.code == -1
    h, n, g0, ps = g.pressure_accumulated(degree, nbins)
    assert n == 6 and np.array_equal(h, total) and total.sum() > 1000
    g0_o, ps_o = oracle_mod.pressure_from_histogram(total.astype(np.float64) / 6, o.N, o.L_eff, o.sigma, dr, degree)
    assert g0 == pytest.approx(g0_o, rel=1e-9) and ps == pytest.approx(ps_o, rel=1e-9)
    # the same fit on a caller's histogram, and one sample == mpmc_pressure_contact
    assert g.pressure_from_histogram(total, 6, dr, degree) == (g0, ps)
    g.pressure_reset()
    g.pressure_accumulate(dr, nbins)
    h1, n1, g1, p1 = g.pressure_accumulated(degree, nbins)
    hc, gc, pc = g.pressure_contact(dr, nbins, degree)
    assert n1 == 1 and np.array_equal(h1, hc) and (g1, p1) == (gc, pc)
    assert_same_state(o, g, fp32)


def test_c3_headline_config_bench_launch_configuration(oracle_mod, torch_cuda):
    """Full size N = 2^20, fp32, NO debug flag: exactly the kernels bench.py times."""
    w = I.CONFIGS["C3"]
    xy, box = I.workload_inputs(w)
    o, g = make_pair(oracle_mod, torch_cuda, w.N, box, w.sigma, w.d, w.n_s, w.seed, True, xy, debug=False)
    assert (g.mx, g.my) == (1152, 998)
    cfg = g.config()
    assert cfg["tiles"] == 148 > cfg["ntx"] * cfg["nty"]       # a mixed tiling: every SM of a B200 gets a tile
    o.sweep(12); g.sweep(12)
    st = assert_same_state(o, g, True, check_mask=False)
    assert st["counts"].sum() == w.N
    assert g.path_sweeps() == (12, 0)                  # the fused tile kernel did them all (crowded cells included)
    att = g.acceptance()[0]
    assert 11.5 * 4.0e6 < att < 12 * 4.2e6
    # a4 at the headline size: C2's bins and the paper's (L382)
    for dr, nbins in [(0.005, 20), (1e-4, 200)]:
        assert np.array_equal(o.contact_histogram(dr, nbins), g.contact_histogram(dr, nbins))


def test_c3_the_config_s_1000_sweeps(oracle_mod, torch_cuda):
    """C3 as BASELINE.json states it — N = 2^20, 1 000 sweeps — on the kernels bench.py times, against the oracle's strip
    program (oracle/strip_omp.cpp: the same Algorithms 2 and 4 on all host cores, identical to the single-thread oracle bit
    for bit: tests/test_strip_baseline.py), which makes 4e9 trial moves affordable."""
    w = I.CONFIGS["C3"]
    xy, box = I.workload_inputs(w)
    from paper_1211_1646_b200.binding import Mpmc
    o = oracle_mod.StripBaseline(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=True)
    g = Mpmc(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=True)
    o.load_positions(xy)
    g.load_positions(torch_cuda.as_tensor(xy, device="cuda"))
    g.sweep(w.sweeps)
    o.sweep(w.sweeps)
    st = assert_same_state(o, g, True, check_mask=False)
    assert st["sweep"] == 1000 and st["counts"].sum() == w.N
    assert g.path_sweeps() == (1000, 0) and g.acceptance()[0] > 3.9e9      # ~4e9 trial moves, all compared through the counters


def test_c3_debug_digest(oracle_mod, torch_cuda):
    w = I.CONFIGS["C3"]
    xy, box = I.workload_inputs(w)
    o, g = make_pair(oracle_mod, torch_cuda, w.N, box, w.sigma, w.d, w.n_s, w.seed, True, xy, debug=True)
    o.sweep(3); g.sweep(3)
    assert_same_state(o, g, True)


@pytest.mark.parametrize("fp32,n", [(True, 512), (False, 256)])
def test_c4_shape_reduced_and_ns8(oracle_mod, torch_cuda, fp32, n):
    # C4's parameters (phi 0.720, d 0.06, n_s 8) on a lattice the oracle finishes in seconds; both precisions
    # (k_tile_sweep<float, 8> and k_tile_sweep<double, 8>)
    xy, box = I.jittered_lattice(n, 0.720, seed=1)
    o, g = make_pair(oracle_mod, torch_cuda, n * n, box, 1.0, 0.06, 8, 1, fp32, xy)
    assert g.config()["tile_slots"] == 2
    o.sweep(8); g.sweep(8)
    assert_same_state(o, g, fp32)
    assert g.path_sweeps() == (8, 0)


def test_c4_full_size_bit_exact(oracle_mod, torch_cuda):
    """BASELINE config C4 at full size (N = 2^24, n_s = 8, fp32, 18.3 M cells, 2538 tiles in 18 waves), NO debug flag:
    two sweeps against the oracle, state compared cell by cell."""
    w = I.CONFIGS["C4"]
    xy, box = I.workload_inputs(w)
    o, g = make_pair(oracle_mod, torch_cuda, w.N, box, w.sigma, w.d, w.n_s, w.seed, True, xy, debug=False)
    assert (g.mx, g.my) == (4596, 3980)
    o.sweep(2); g.sweep(2)
    st = assert_same_state(o, g, True, check_mask=False)
    assert st["counts"].sum() == w.N and g.path_sweeps() == (2, 0)


def melted_by_the_oracle(oracle_mod, n, phi, d, w_target=0.0, fp32=True):
    """Reading A15: the method itself with a fixed preparation seed until attempted >= 100 N.  The ORACLE melts: no
    oracle input ever comes from the CUDA path."""
    xy0, box = I.jittered_lattice(n, phi, seed=1)
    pre = oracle_mod.Oracle(n * n, box, 1.0, d, 4, 999, fp32=fp32, w_target=w_target)
    pre.load_positions(xy0)
    while pre.acceptance()[0] < 100 * n * n:
        pre.sweep(10)
    return pre.get_positions(), box


def test_c5_dilute_fluid_reduced(oracle_mod, torch_cuda):
    # C5's parameters (phi 0.30, d 0.5, w = sigma) on 256^2 disks, 60 sweeps with the accept masks compared
    n = 256
    xy, box = melted_by_the_oracle(oracle_mod, n, 0.30, 0.5)
    o, g = make_pair(oracle_mod, torch_cuda, n * n, box, 1.0, 0.5, 4, 1, True, xy)
    assert g.config()["tile_slots"] == 2
    for _ in range(6):
        o.sweep(10); g.sweep(10)
        st = assert_same_state(o, g, True)
    assert st["counts"].max() >= 2 and (st["counts"] == 0).mean() > 0.5
    assert g.path_sweeps() == (60, 0)
    att, acc, rb, ro = g.acceptance()
    assert rb / att > 0.3           # boundary-crossing rejections dominate at d = 0.5 (config C5)


def test_c5_full_size(oracle_mod, torch_cuda):
    """BASELINE config C5 at its configured size (N = 2^20, phi = 0.30, 1780 x 1540 cells), NO debug flag: the launch
    configuration bench.py --workload C5 times (compacting variant of the tile kernel)."""
    w = I.CONFIGS["C5"]
    xy, box = melted_by_the_oracle(oracle_mod, w.n_side, w.phi, w.d)
    o, g = make_pair(oracle_mod, torch_cuda, w.N, box, w.sigma, w.d, w.n_s, w.seed, True, xy, debug=False)
    assert (g.mx, g.my) == (1780, 1540)
    assert g.config()["tile_slots"] == 2
    o.sweep(10); g.sweep(10)
    st = assert_same_state(o, g, True, check_mask=False)
    assert g.path_sweeps() == (10, 0)
    assert st["counts"].sum() == w.N and (st["counts"] == 0).mean() > 0.6 and st["counts"].max() >= 2
    att, acc, rb, ro = g.acceptance()
    assert rb / att > 0.3


@pytest.mark.parametrize("fp32", [True, False])
def test_dilute_fluid_with_three_per_cell(oracle_mod, torch_cuda, fp32):
    # C5's density and displacement at a cell width just under 1.15 sigma: still the 2-slot tile kernel (0.48 disks per
    # cell: most queue entries are dropped as empty), and cells with THREE disks do occur — occupancy queues x the list of
    # crowded cells
    n = 256
    xy, box = melted_by_the_oracle(oracle_mod, n, 0.30, 0.5, w_target=1.12, fp32=fp32)
    o, g = make_pair(oracle_mod, torch_cuda, n * n, box, 1.0, 0.5, 4, 1, fp32, xy, w_target=1.12)
    assert g.config()["tile_slots"] == 2
    seen3, sweeps_with3 = False, 0
    for _ in range(8):
        o.sweep(5); g.sweep(5)
        st = assert_same_state(o, g, fp32)
        has3 = st["counts"].max() >= 3
        seen3 |= has3; sweeps_with3 += int(has3)
    assert seen3 and sweeps_with3 >= 2
    assert g.path_sweeps() == (40, 0)                  # the tile kernel carried the crowded cells itself


@pytest.mark.parametrize("fp32", [False, True])
def test_three_per_cell_with_two_register_slots(oracle_mod, torch_cuda, fp32):
    # w ~ 1.13 sigma keeps the NF = 2 kernel (w < 1.15 sigma) while cells with 3 disks do occur: exercises the
    # path that re-reads slots 2, 3 of crowded neighbours inside the move loop
    xy, box = I.jittered_lattice(64, 0.50, seed=6)
    o, g = make_pair(oracle_mod, torch_cuda, 4096, box, 1.0, 0.3, 4, 8, fp32, xy, w_target=1.12)
    assert 1.12 <= g.wx < 1.15 and 1.12 <= g.wy < 1.15
    seen3 = False
    for _ in range(10):
        o.sweep(20); g.sweep(20)
        st = assert_same_state(o, g, fp32)
        seen3 |= st["counts"].max() >= 3
    assert seen3
    tile, general = g.path_sweeps()
    assert tile + general == 200 and tile > 0          # crowded cells carried by the tile kernel's shared-memory list


@pytest.mark.parametrize("fp32", [False, True])
def test_tile_kernel_hands_over_when_too_many_cells_are_crowded(oracle_mod, torch_cuda, fp32):
    # a denser system at the same cell width: more than 256 cells hold 3 disks, so the tile kernel returns at once
    # and the general persistent kernel runs the sweeps (and the tile kernel resumes if the state thins out)
    xy, box = I.jittered_lattice(192, 0.70, seed=9)
    o, g = make_pair(oracle_mod, torch_cuda, 192 * 192, box, 1.0, 0.2, 4, 5, fp32, xy, w_target=1.135)
    assert 1.135 <= g.wx < 1.15 and 1.135 <= g.wy < 1.15
    most = 0
    for _ in range(4):
        o.sweep(10); g.sweep(10)
        st = assert_same_state(o, g, fp32)
        most = max(most, int((st["counts"] >= 3).sum()))
    tile, general = g.path_sweeps()
    assert tile + general == 40
    assert general > 0 and most > 256


@pytest.mark.parametrize("n,phi", [(14, 0.5), (24, 0.6), (50, 0.7), (98, 0.65),
                                   (14, 0.3), (26, 0.38), (50, 0.33), (98, 0.4), (150, 0.25)])    # dilute: most cells empty
def test_tile_kernel_uneven_tilings(oracle_mod, torch_cuda, n, phi):
    # box sizes that do not divide evenly into tiles (tiles of different widths, many tiny tiles, few large ones)
    xy, box = I.jittered_lattice(n, phi, seed=n)
    o, g = make_pair(oracle_mod, torch_cuda, n * n, box, 1.0, 0.15 if phi >= 0.5 else 0.4, 4, n, True, xy)
    cfg = g.config()
    assert cfg["tile_slots"] == 2 and cfg["tiles"] >= cfg["ntx"] * cfg["nty"] > 1      # (mixed tilings: some rows hold ntx + 1)
    for k in (1, 2, 7):
        o.sweep(k); g.sweep(k)
        assert_same_state(o, g, True)
    assert g.path_sweeps() == (10, 0)


@pytest.mark.parametrize("fp32", [False, True])
def test_mixed_tiling_two_tile_shapes(oracle_mod, torch_cuda, fp32):
    # a grid whose best tiling has rows of a and rows of a + 1 tiles (tile_box): accept masks compared over 15 sweeps
    xy, box = I.jittered_lattice(200, 0.68, seed=31)
    o, g = make_pair(oracle_mod, torch_cuda, 200 * 200, box, 1.0, 0.12, 4, 4, fp32, xy)
    cfg = g.config()
    assert cfg["tile_slots"] == 2 and cfg["tiles"] > cfg["ntx"] * cfg["nty"]
    for k in (1, 4, 10):
        o.sweep(k); g.sweep(k)
        assert_same_state(o, g, fp32)
    assert g.path_sweeps() == (15, 0)


@pytest.mark.parametrize("n_s", [4, 8])
def test_dilute_system_fp64(oracle_mod, torch_cuda, n_s):
    xy, box = I.jittered_lattice(60, 0.35, seed=8)
    o, g = make_pair(oracle_mod, torch_cuda, 3600, box, 1.0, 0.4, n_s, 2, False, xy)
    assert g.config()["tile_slots"] == 2
    o.sweep(12); g.sweep(12)
    assert_same_state(o, g, False)
    assert g.path_sweeps() == (12, 0)


@pytest.mark.parametrize("fp32", [False, True])
def test_paper_cell_regime_w_1p4(oracle_mod, torch_cuda, fp32):
    # cell width just under sqrt(2) sigma, n_max = 4 fully used (L152); 4-slot tile kernel
    xy, box = I.jittered_lattice(128, 0.698, seed=2)
    o, g = make_pair(oracle_mod, torch_cuda, 128 * 128, box, 1.0, 0.16, 4, 3, fp32, xy, w_target=1.40)
    assert g.wx >= 1.40 and g.wx < math.sqrt(2)
    o.sweep(25); g.sweep(25)
    st = assert_same_state(o, g, fp32)
    assert st["counts"].max() >= 3


@pytest.mark.parametrize("fp32", [False, True])
@pytest.mark.parametrize("n_s", [4, 3])
def test_paper_regime_with_disc_proposal(oracle_mod, torch_cuda, fp32, n_s):
    # SURVEY.md §8(f).1 in full: w just under sqrt(2) sigma, disc-shaped displacement of radius 0.16 sigma (L190, L358)
    w = I.CONFIGS["P256"]
    xy, box = I.workload_inputs(w)
    o, g = make_pair(oracle_mod, torch_cuda, w.N, box, w.sigma, w.d, n_s, 7, fp32, xy, w_target=w.w_target, disc=True)
    assert g.wx >= 1.40 and g.wx < math.sqrt(2)
    o.sweep(20); g.sweep(20)
    st = assert_same_state(o, g, fp32)
    assert st["counts"].max() >= 3
    assert g.path_sweeps() == ((20, 0) if n_s == 4 else (0, 20))     # 4-slot tile kernel for n_s = 4, else the general kernel


@pytest.mark.parametrize("n,phi,disc", [(20, 0.5, False), (34, 0.66, True), (70, 0.698, False), (126, 0.6, True)])
def test_four_slot_tile_kernel_uneven_tilings(oracle_mod, torch_cuda, n, phi, disc):
    # w = 1.4 sigma on boxes that do not divide evenly into tiles; both proposals
    xy, box = I.jittered_lattice(n, phi, seed=n)
    o, g = make_pair(oracle_mod, torch_cuda, n * n, box, 1.0, 0.16, 4, n + 1, True, xy, w_target=1.40, disc=disc)
    for k in (1, 3, 6):
        o.sweep(k); g.sweep(k)
        assert_same_state(o, g, True)
    assert sum(g.path_sweeps()) == 10


@pytest.mark.parametrize("pshuf,sshuf", [(False, True), (True, False), (False, False)])
@pytest.mark.parametrize("w_target,n_s", [(0.0, 4), (1.40, 4), (1.40, 6)])      # 2-slot tile, 4-slot tile, general kernel
def test_ablation_switches(oracle_mod, torch_cuda, pshuf, sshuf, w_target, n_s):
    # PAPER.md section 2.4 / Table 1: particle shuffle and checkerboard-set shuffle switched off
    xy, box = I.jittered_lattice(64, 0.66, seed=12)
    o, g = make_pair(oracle_mod, torch_cuda, 4096, box, 1.0, 0.2, n_s, 3, True, xy, w_target=w_target,
                     particle_shuffle=pshuf, set_shuffle=sshuf)
    o.sweep(12); g.sweep(12)
    assert_same_state(o, g, True)


def test_disc_proposal_at_unit_cell_width(oracle_mod, torch_cuda):
    xy, box = I.jittered_lattice(64, 0.6, seed=3)
    o, g = make_pair(oracle_mod, torch_cuda, 4096, box, 1.0, 0.2, 4, 9, True, xy, disc=True)
    o.sweep(15); g.sweep(15)
    assert_same_state(o, g, True)
    assert g.path_sweeps() == (15, 0)                  # the 4-slot tile kernel serves the disc proposal at any width


@pytest.mark.parametrize("N,box,xy", [
    (1, (2.6, 2.6), [[0.3, 0.4]]),
    (2, (2.6, 2.9), [[0.5, 0.5], [1.8, 1.9]]),                 # mx = my = 2: neighbour at two image offsets
    (3, (4.3, 4.5), [[0.5, 0.5], [2.0, 2.0], [3.5, 0.9]]),
])
@pytest.mark.parametrize("fp32", [False, True])
def test_tiny_systems(oracle_mod, torch_cuda, N, box, xy, fp32):
    xy = np.array(xy, dtype=np.float64)
    o, g = make_pair(oracle_mod, torch_cuda, N, box, 1.0, 0.4, 4, 9, fp32, xy)
    for _ in range(5):
        o.sweep(40); g.sweep(40)
        assert_same_state(o, g, fp32)


@pytest.mark.parametrize("n_s", [0, 1, 7, 32])
def test_moves_per_cell_range(oracle_mod, torch_cuda, n_s):
    xy, box = I.jittered_lattice(32, 0.6, seed=4)
    o, g = make_pair(oracle_mod, torch_cuda, 1024, box, 1.0, 0.2, n_s, 5, False, xy)
    o.sweep(20); g.sweep(20)
    assert_same_state(o, g, False)
    assert g.acceptance()[0] == o.acceptance()[0]
    if n_s == 0:
        assert g.acceptance() == (0, 0, 0, 0)


def test_seed_and_high_sweep_words(oracle_mod, torch_cuda):
    xy, box = I.jittered_lattice(32, 0.6, seed=4)
    seed = 0xDEADBEEF12345678
    o, g = make_pair(oracle_mod, torch_cuda, 1024, box, 1.0, 0.2, 4, seed, True, xy)
    o.sweep(5); g.sweep(5)
    assert_same_state(o, g, True)


def test_two_live_contexts_with_different_tilings(oracle_mod, torch_cuda):
    """Two contexts of the SAME kernel instantiation with different tilings and shared-memory sizes, sweeps interleaved:
    the dynamic shared-memory limit is a property of the kernel function, so the second create must not undo the first."""
    big = I.jittered_lattice(256, 0.70, seed=1)
    small = I.jittered_lattice(32, 0.6, seed=4)
    ob, gb = make_pair(oracle_mod, torch_cuda, 256 * 256, big[1], 1.0, 0.1, 4, 1, True, big[0])
    os_, gs = make_pair(oracle_mod, torch_cuda, 1024, small[1], 1.0, 0.2, 4, 5, True, small[0])
    assert gb.config()["tile_smem"] > 4 * gs.config()["tile_smem"] > 0
    for k in (1, 3, 2):
        gb.sweep(k); gs.sweep(k); ob.sweep(k); os_.sweep(k)
        gs.sweep(1); gb.sweep(1); os_.sweep(1); ob.sweep(1)
    assert_same_state(ob, gb, True)
    assert_same_state(os_, gs, True)
    assert gb.path_sweeps() == (9, 0) and gs.path_sweeps() == (9, 0)


def test_two_live_resident_contexts_and_a_tiled_one(oracle_mod, torch_cuda):
    """Two contexts on the SAME instantiation of the cluster-resident kernel with different tile sizes (hence different
    dynamic shared memory: a property of the kernel function) and one on the tile kernel, sweeps interleaved on their own
    streams."""
    a = I.jittered_lattice(96, 0.70, seed=1)
    b = I.jittered_lattice(32, 0.6, seed=4)
    c = I.jittered_lattice(64, 0.65, seed=9)
    oa, ga = make_pair(oracle_mod, torch_cuda, 96 * 96, a[1], 1.0, 0.1, 4, 1, True, a[0], resident=True)
    ob, gb = make_pair(oracle_mod, torch_cuda, 1024, b[1], 1.0, 0.2, 4, 5, True, b[0], resident=True)
    oc, gc = make_pair(oracle_mod, torch_cuda, 4096, c[1], 1.0, 0.15, 4, 6, True, c[0], resident=False)
    assert ga.config()["resident_smem"] > 4 * gb.config()["resident_smem"] > 0 and gc.config()["resident_ctas"] == 0
    for k in (1, 3, 2):
        ga.sweep(k); gb.sweep(k); gc.sweep(k); oa.sweep(k); ob.sweep(k); oc.sweep(k)
        gb.sweep(1); gc.sweep(1); ga.sweep(1); ob.sweep(1); oc.sweep(1); oa.sweep(1)
    for o, g in ((oa, ga), (ob, gb), (oc, gc)):
        assert_same_state(o, g, True)
        assert g.path_sweeps() == (9, 0)


def test_debug_shift_rejects_a_shift_of_a_cell_width(oracle_mod, torch_cuda):
    from paper_1211_1646_b200.binding import MpmcError
    xy, box = I.jittered_lattice(32, 0.6, seed=4)
    o, g = make_pair(oracle_mod, torch_cuda, 1024, box, 1.0, 0.2, 4, 5, True, xy)
    with pytest.raises(MpmcError) as e:
        g.shift(0, g.wx)               # the pull form takes entrants from one neighbour only: delta < w
    assert e.value.code == -1
    g.shift(0, 0.49 * g.wx); o.shift(0, 0.49 * o.wx)
    assert_same_state(o, g, True)


def test_errors_on_device(oracle_mod, torch_cuda):
    torch = torch_cuda
    from paper_1211_1646_b200.binding import Mpmc, MpmcError
    g = Mpmc(2, (4.4, 4.4), 1.0, 0.1, 4, 1)
    with pytest.raises(MpmcError) as e:
        g.sweep(1)
    assert e.value.code == -7
    with pytest.raises(MpmcError) as e:
        g.load_positions(torch.tensor([[1.0, 1.0], [1.5, 1.0]], dtype=torch.float64, device="cuda"))
    assert e.value.code == -4
    with pytest.raises(MpmcError):
        g.load_positions(torch.tensor([[1.0, 1.0], [float("nan"), 1.0]], dtype=torch.float64, device="cuda"))
    with pytest.raises(MpmcError):
        g.load_positions(torch.tensor([[0.1, 1.0], [4.3, 1.0]], dtype=torch.float64, device="cuda"))   # across the edge
    g.load_positions(torch.tensor([[1.0, 1.0], [2.0, 1.0]], dtype=torch.float64, device="cuda"))       # r = sigma: fine
    g.sweep(3)
    assert g.acceptance()[0] > 0
    with pytest.raises(MpmcError) as e:
        Mpmc(2, (1.9, 4.4), 1.0, 0.1, 4, 1)
    assert e.value.code == -2
    # five disks forced into one wide cell -> overflow reported at load
    g5 = Mpmc(5, (6.4, 6.4), 1.0, 0.1, 4, 1, w_target=3.0)
    pts = torch.tensor([[0.2, 0.2], [1.4, 0.2], [2.6, 0.2], [0.2, 1.4], [1.4, 1.4]], dtype=torch.float64, device="cuda")
    with pytest.raises(MpmcError) as e:
        g5.load_positions(pts)
    assert e.value.code == -5


def test_overlap_free_and_conserved_at_full_size(torch_cuda):
    """Properties that hold at any size, at the headline size and in the bench launch configuration."""
    torch = torch_cuda
    from scipy.spatial import cKDTree
    from paper_1211_1646_b200.binding import Mpmc
    w = I.CONFIGS["C3"]
    xy, box = I.workload_inputs(w)
    g = Mpmc(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=True)
    g.load_positions(torch.as_tensor(xy, device="cuda"))
    g.sweep(200)
    p = g.get_positions().cpu().numpy()
    assert np.isfinite(p).all() and p.shape == (w.N, 2)
    Le = np.array(g.L_eff)
    assert (p >= 0).all() and (p < Le).all()
    tree = cKDTree(np.minimum(p, np.nextafter(Le, 0)), boxsize=Le)
    dmin = tree.query(p, k=2)[0][:, 1].min()
    # fp32 locals: the overlap test is made in the mover's frame and two cells' frames differ by an ulp, so seen from
    # the unpacked doubles r^2 >= sigma^2 (1 - 4 eps_P), eps_P = 2^-23
    assert dmin >= math.sqrt(1.0 - 4 * float(np.finfo(np.float32).eps)) and dmin < 1.001
    st = g.debug_state()
    assert st["counts"].sum() == w.N and st["counts"].max() <= 4 and st["sweep"] == 200
    used = np.arange(4)[None, :] < st["counts"][:, None]
    assert np.array_equal(np.sort(st["ids"][used]), np.arange(w.N, dtype=np.uint32))
    att, acc, rb, ro = g.acceptance()
    assert att == acc + rb + ro and 0.2 < acc / att < 0.9
