"""Bookkeeping and geometry pins for the oracle (CPU only).

Fixed from outside the oracle: the disk count is conserved and ids stay a permutation,
n <= n_max = 4 (L152), every local coordinate lies in (0, w] (Alg. 4 lines 10/21), every configuration is
overlap-free — checked here with an independent periodic KD-tree in double on the unpacked global
coordinates — a pure grid shift leaves every global position where it was (L350), and a disk only moves
when its move was accepted.
"""
import math

import numpy as np
import pytest
from scipy.spatial import cKDTree

from paper_1211_1646_b200 import inputs as I


def min_pair_distance(xy, L):
    xy = np.mod(xy, np.asarray(L))
    xy = np.minimum(xy, np.nextafter(np.asarray(L), 0))
    tree = cKDTree(xy, boxsize=np.asarray(L))
    d, _ = tree.query(xy, k=2)
    return d[:, 1].min()


def periodic_delta(a, b, L):
    d = a - b
    return d - np.asarray(L) * np.round(d / np.asarray(L))


def check_state(o, st):
    n = st["counts"]
    assert n.sum() == o.N
    assert n.max() <= 4
    used = np.arange(4)[None, :] < n[:, None]
    ids = st["ids"][used]
    assert np.array_equal(np.sort(ids), np.arange(o.N, dtype=np.uint32))
    assert np.all(st["ids"][~used] == 0xFFFFFFFF)
    lx = st["slab"][..., 0][used]
    ly = st["slab"][..., 1][used]
    assert np.all(lx > 0) and np.all(lx <= o.real(o.wx))
    assert np.all(ly > 0) and np.all(ly <= o.real(o.wy))


@pytest.mark.parametrize("fp32", [False, True])
def test_c1_invariants_every_sweep(oracle_mod, fp32):
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    o = oracle_mod.Oracle(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=fp32)
    assert (o.mx, o.my) == (86, 74)
    assert o.wx >= w.sigma and o.wy >= w.sigma
    o.load_positions(xy)
    eps = float(np.finfo(np.float32 if fp32 else np.float64).eps)     # r^2 >= sigma^2 (1 - 4 eps_P)
    got = o.get_positions()
    assert np.abs(periodic_delta(got, xy, o.L_eff)).max() < (2e-4 if fp32 else 1e-12)
    last = o.acceptance()
    for sweep in range(30):
        o.sweep(1)
        st = o.debug_state()
        assert st["sweep"] == sweep + 1
        check_state(o, st)
        a = o.acceptance()
        assert a[0] == a[1] + a[2] + a[3]
        # attempted = n_s per non-empty active cell (reading A10): every non-empty cell once per sweep...
        assert 0 < a[0] - last[0] <= w.n_s * o.M
        last = a
        pos = o.get_positions()
        assert np.all(pos >= 0) and np.all(pos[:, 0] < o.L_eff[0]) and np.all(pos[:, 1] < o.L_eff[1])
        # (the unpacked doubles carry their own rounding, ~1e-14 at X ~ 90, which only matters in fp64)
        assert min_pair_distance(pos, o.L_eff) >= w.sigma * math.sqrt(1 - 4 * eps) - (0 if fp32 else 1e-12)
    assert last[1] > 0 and last[2] > 0 and last[3] > 0


def test_dense_fp32_hard_core_within_four_eps(oracle_mod):
    """The same pin where it bites: phi = 0.716 (config C3's density), fp32, where many pairs sit at r ~ sigma.  The
    overlap test is made in the mover's cell frame in fp32; seen from unpacked double coordinates the frames of two
    cells differ by an ulp, hence r^2 >= sigma^2 (1 - 4 eps_P) and not r >= sigma."""
    xy, box = I.jittered_lattice(64, 0.716, seed=3)
    o = oracle_mod.Oracle(4096, box, 1.0, 0.08, 4, 3, fp32=True)
    o.load_positions(xy)
    eps = float(np.finfo(np.float32).eps)
    for _ in range(20):
        o.sweep(5)
        d = min_pair_distance(o.get_positions(), o.L_eff)
        assert d >= math.sqrt(1 - 4 * eps) and d < 1.001          # close pairs do exist: the pin is not vacuous


def test_attempted_counts_nonempty_active_cells(oracle_mod):
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    o = oracle_mod.Oracle(w.N, box, w.sigma, w.d, w.n_s, w.seed)
    o.load_positions(xy)
    total = 0
    for q in range(4):
        n = o.debug_state()["counts"].reshape(o.my, o.mx)
        active = n[(q >> 1)::2, (q & 1)::2]
        total += w.n_s * int((active > 0).sum())
        o.sub_sweep(q)
        assert o.acceptance()[0] == total


def test_only_accepted_moves_move_disks(oracle_mod):
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    o = oracle_mod.Oracle(w.N, box, w.sigma, w.d, w.n_s, w.seed)
    o.load_positions(xy)
    before = o.debug_state()
    o.sub_sweep(0)
    after = o.debug_state()
    assert np.array_equal(before["ids"], after["ids"]) and np.array_equal(before["counts"], after["counts"])
    moved_cells = np.any(before["slab"] != after["slab"], axis=(1, 2))
    x = np.arange(o.M) % o.mx
    y = np.arange(o.M) // o.mx
    in_set_a = (x % 2 == 0) & (y % 2 == 0)
    assert not np.any(moved_cells & ~in_set_a)               # eq. 1: only set a is active
    assert np.array_equal(moved_cells, after["accept_mask"] != 0)
    assert np.all(after["accept_mask"] < (1 << w.n_s))
    acc = o.acceptance()
    assert acc[1] == sum(bin(int(m)).count("1") for m in after["accept_mask"])
    # no displacement exceeds d per coordinate times the number of moves of that disk
    disp = np.abs(after["slab"] - before["slab"])
    assert disp.max() <= w.d * w.n_s


@pytest.mark.parametrize("fp32", [False, True])
@pytest.mark.parametrize("direction", [0, 1, 2, 3])
def test_shift_keeps_global_positions(oracle_mod, fp32, direction):
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    o = oracle_mod.Oracle(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=fp32)
    o.load_positions(xy)
    p0 = o.get_positions()
    s0 = o.debug_state()
    delta = 0.37 * (o.wx if direction < 2 else o.wy)
    o.shift(direction, delta)
    s1 = o.debug_state()
    check_state(o, s1)
    p1 = o.get_positions()
    assert np.abs(periodic_delta(p1, p0, o.L_eff)).max() < (1e-5 if fp32 else 1e-13)
    axis = 0 if direction < 2 else 1
    sign = 1.0 if direction % 2 == 0 else -1.0
    expect = (sign * float(o.real(delta))) % o.L_eff[axis]
    assert s1["origin"][axis] == pytest.approx(expect, abs=1e-15)
    assert s1["origin"][1 - axis] == 0.0
    # some disks changed cell, and the cell counts moved accordingly
    assert not np.array_equal(s0["counts"], s1["counts"])
    # +f shift: local coordinates of stayers decrease by delta (disks are translated by -f*delta, L303/L350)
    c = np.flatnonzero((s0["counts"] == 1) & (s1["counts"] == 1) & (s0["ids"][:, 0] == s1["ids"][:, 0]))
    assert len(c) > 100
    dl = s1["slab"][c, 0, axis].astype(np.float64) - s0["slab"][c, 0, axis].astype(np.float64)
    assert np.allclose(dl, -sign * float(o.real(delta)), atol=2e-6 if fp32 else 1e-15)


def test_slot_order_after_shift_is_stayers_then_entrants(oracle_mod):
    # 4x4 cells of width 1.1; all four disks sit in cell row 0.  A +x shift by 0.3 makes A (cell 1, local
    # 0.05) and C (cell 2, local 0.10) leave to the cell on their left; B and D stay.  Reading A13 / Alg. 4
    # lines 7-27: new slot order = stayers (old slot order) then entrants — NOT ascending id.
    box = (4.4, 4.4)
    xy = np.array([[1.15, 0.05],    # id 0 = A
                   [0.70, 1.00],    # id 1 = B
                   [2.30, 0.05],    # id 2 = C
                   [1.90, 1.00]])   # id 3 = D
    o = oracle_mod.Oracle(4, box, 1.0, 0.1, 4, 7)
    assert (o.mx, o.my) == (4, 4)
    o.load_positions(xy)
    st = o.debug_state()
    assert list(st["ids"].reshape(4, 4, 4)[0, 1][:2]) == [0, 3]      # load order: ascending id
    o.shift(0, 0.3)
    st = o.debug_state()
    ids = st["ids"].reshape(4, 4, 4)
    cnt = st["counts"].reshape(4, 4)
    assert cnt[0, 0] == 2 and list(ids[0, 0][:2]) == [1, 0]          # B stays, then A enters
    assert cnt[0, 1] == 2 and list(ids[0, 1][:2]) == [3, 2]          # D stays, then C enters
    assert cnt.sum() == 4
    slab = st["slab"].reshape(4, 4, 4, 2)
    assert slab[0, 0, 1, 0] == pytest.approx(0.05 - 0.3 + 1.1, abs=1e-12)   # A: l' = l - delta, then + w
    assert slab[0, 0, 0, 0] == pytest.approx(0.70 - 0.3, abs=1e-12)
    assert np.allclose(o.get_positions(), xy, atol=1e-14)
    # and back: a -x shift by the same amount
    o.shift(1, 0.3)
    st = o.debug_state()
    ids = st["ids"].reshape(4, 4, 4)
    assert list(ids[0, 0][:1]) == [1] and list(ids[0, 1][:2]) == [3, 0] and list(ids[0, 2][:1]) == [2]
    assert np.allclose(o.get_positions(), xy, atol=1e-14)


def test_load_rejects_overlap_and_out_of_box(oracle_mod):
    box = (4.4, 4.4)
    o = oracle_mod.Oracle(2, box, 1.0, 0.1, 4, 1)
    with pytest.raises(oracle_mod.OracleError) as e:
        o.load_positions(np.array([[1.0, 1.0], [1.5, 1.0]]))
    assert e.value.code == -4
    with pytest.raises(oracle_mod.OracleError):
        o.load_positions(np.array([[1.0, 1.0], [5.5, 1.0]]))
    with pytest.raises(oracle_mod.OracleError):
        o.load_positions(np.array([[1.0, 1.0], [float("nan"), 1.0]]))
    # touching across the periodic boundary is an overlap too
    with pytest.raises(oracle_mod.OracleError):
        o.load_positions(np.array([[0.1, 1.0], [4.3, 1.0]]))
    o.load_positions(np.array([[1.0, 1.0], [2.0, 1.0]]))          # r = sigma exactly: not an overlap (A4)
    with pytest.raises(oracle_mod.OracleError):
        oracle_mod.Oracle(2, (1.9, 4.4), 1.0, 0.1, 4, 1)          # mx < 2
    with pytest.raises(oracle_mod.OracleError):
        oracle_mod.Oracle(2, box, 1.0, 0.1, 4, 1).sweep(1)        # nothing loaded


def test_geometry_of_baseline_configs(oracle_mod):
    # (mx, my) per config
    want = {"C1": (86, 74), "C2": (290, 252), "C3": (1152, 998), "C4": (4596, 3980), "C5": (1780, 1540)}
    for name, (mx, my) in want.items():
        w = I.CONFIGS[name]
        box = I.box_for(w.n_side, w.phi, w.sigma)
        m = [2 * math.floor(box[a] / 2.0) for a in range(2)]
        assert (m[0], m[1]) == (mx, my)
        if w.N <= 65536:
            o = oracle_mod.Oracle(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=w.fp32)
            assert (o.mx, o.my) == (mx, my)
            assert 1.0 <= o.wx < math.sqrt(2) and 1.0 <= o.wy < math.sqrt(2)


def test_deterministic_and_seed_dependent(oracle_mod):
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    runs = []
    for seed in (1, 1, 2):
        o = oracle_mod.Oracle(w.N, box, w.sigma, w.d, w.n_s, seed)
        o.load_positions(xy)
        o.sweep(5)
        runs.append((o.get_positions(), o.acceptance(), o.debug_state()["digest"]))
    assert np.array_equal(runs[0][0], runs[1][0]) and runs[0][1:] == runs[1][1:]
    assert not np.array_equal(runs[0][0], runs[2][0]) and runs[0][2] != runs[2][2]
    # k sweeps at once == k single sweeps
    o = oracle_mod.Oracle(w.N, box, w.sigma, w.d, w.n_s, 1)
    o.load_positions(xy)
    for _ in range(5):
        o.sweep(1)
    assert np.array_equal(o.get_positions(), runs[0][0])


# ---- ablation switches of PAPER.md section 2.4 / Table 1 (L114-142) -------------------------------------------------
def test_without_particle_shuffle_the_first_move_acts_on_slot_zero(oracle_mod):
    """Two disks in one cell, n_s = 1: without the particle shuffle (L187 left out) the single move of a sub-sweep always
    acts on slot 0 = the lower id (slots ascend by id at load, A13); with it, slot 1 goes first about half the time."""
    box, xy = (2.6, 2.6), np.array([[0.25, 0.30], [1.20, 1.25]])          # w = 1.3: both in cell (0, 0)
    moved_second = {True: 0, False: 0}
    for shuffle in (False, True):
        for seed in range(200):
            o = oracle_mod.Oracle(2, box, 1.0, 0.05, 1, seed, w_target=1.3, particle_shuffle=shuffle)
            assert (o.mx, o.my) == (2, 2)
            o.load_positions(xy)
            o.sub_sweep(0)                                                    # set a holds cell (0, 0)
            p = o.get_positions()
            assert np.all(o.debug_state()["counts"].reshape(2, 2) == [[2, 0], [0, 0]])
            if not np.array_equal(p[1], xy[1]):
                moved_second[shuffle] += 1
    assert moved_second[False] == 0
    assert 50 < moved_second[True] < 150          # about half of the accepted first moves (acceptance < 1)


def test_without_set_shuffle_the_sets_run_in_order_abcd(oracle_mod):
    """set_shuffle = False: a sweep equals sub-sweeps a, b, c, d in that order followed by the drawn shift (composed from
    the single-piece hooks); with the shuffle some sweep differs from that composition."""
    xy, box = I.jittered_lattice(12, 0.55, seed=3)
    differs = False
    for shuffle in (False, True):
        # compose sweep 0 by hand on a fresh copy
        a = oracle_mod.Oracle(144, box, 1.0, 0.2, 4, 5, set_shuffle=shuffle)
        b = oracle_mod.Oracle(144, box, 1.0, 0.2, 4, 5, set_shuffle=shuffle)
        a.load_positions(xy); b.load_positions(xy)
        a.sweep(1)
        order, direction, word = oracle_mod.sweep_draws(5, 0)
        for q in (0, 1, 2, 3):
            b.sub_sweep(q)
        w_axis = b.wx if direction < 2 else b.wy
        b.shift(direction, (0.5 * w_axis) * (word * 2.0 ** -32))
        same = np.array_equal(a.get_positions(), b.get_positions())
        if shuffle:
            differs |= (order != [0, 1, 2, 3]) and not same
        else:
            assert same
    assert differs or oracle_mod.sweep_draws(5, 0)[0] == [0, 1, 2, 3]


# ---- ablation "disks may leave their cell" (section 2.4 pitfall 1, L118-122; oracle only) ----------------------
def test_leave_cell_ablation_keeps_the_books_and_the_hard_core(oracle_mod):
    """With the restriction of L118 lifted a move is never rejected for leaving the cell: the disk is handed to the cell
    it lands in (appended to that list, L123) after a Metropolis test made THERE.  Fixed from outside: the disk count and
    the ids are conserved, every local lies in (0, w], no overlap ever appears (independent KD-tree), no boundary
    rejection is counted, and more moves are accepted than with the restriction."""
    xy, box = I.jittered_lattice(64, 0.6, seed=4)
    for fp32 in (False, True):
        o = oracle_mod.Oracle(4096, box, 1.0, 0.3, 4, 9, fp32=fp32, leave_cell=True)
        ref = oracle_mod.Oracle(4096, box, 1.0, 0.3, 4, 9, fp32=fp32)
        o.load_positions(xy); ref.load_positions(xy)
        eps = float(np.finfo(np.float32 if fp32 else np.float64).eps)
        for _ in range(10):
            o.sweep(4); ref.sweep(4)
            check_state(o, o.debug_state())
            assert min_pair_distance(o.get_positions(), o.L_eff) >= math.sqrt(1 - 4 * eps) - (0 if fp32 else 1e-12)
        a, b = o.acceptance(), ref.acceptance()
        assert a[0] == a[1] + a[3] and a[2] == 0 and b[2] > 0
        assert a[1] / a[0] > b[1] / b[0] + 0.03
        moved = np.abs(periodic_delta(o.get_positions(), xy, o.L_eff)).max()
        assert moved > 1.0                                 # disks do travel across cells


def test_leave_cell_ablation_isolated_disk_walks_freely(oracle_mod):
    """N = 1: nothing to overlap with and no boundary to stop at, so every move is accepted and the disk performs a free
    random walk: <|dr|^2> = T * 2 d^2 / 3 after T moves of U[-d, d]^2.  A wrong translation when the disk changes cell (a
    lost or doubled +-w) would add jumps of a cell width and inflate this several-fold."""
    L, d, n_s, sweeps = (6.4, 6.6), 0.4, 4, 30
    msd, moves = [], []
    for seed in range(120):
        o = oracle_mod.Oracle(1, L, 1.0, d, n_s, 1000 + seed, leave_cell=True)
        o.load_positions(np.array([[3.1, 3.3]]))
        prev, total = o.get_positions()[0], np.zeros(2)
        for _ in range(sweeps):
            o.sweep(1)
            p = o.get_positions()[0]
            total += periodic_delta(p, prev, o.L_eff)          # at most n_s d = 1.6 per sweep, under L/2
            prev = p
        a = o.acceptance()
        # every attempt is accepted; their number per sweep is no longer n_s: a cell update ends when its disk has left, and
        # a disk that lands in a cell whose set runs later in the sweep is moved again (the state-dependent schedule the
        # paper warns of, L118-122)
        assert a[0] == a[1] and 0.5 * sweeps * n_s < a[0] < 2 * sweeps * n_s
        msd.append((total ** 2).sum()); moves.append(a[1])
    want = np.mean(moves) * 2 * d * d / 3
    assert abs(np.mean(msd) / want - 1) < 0.25, (np.mean(msd), want)


def test_leave_cell_ablation_coincides_with_the_method_until_a_disk_leaves(oracle_mod):
    # same seed: the two chains are the same move for move until the first move that leaves its cell
    o = oracle_mod.Oracle(1, (6.4, 6.6), 1.0, 0.05, 4, 5, leave_cell=True)
    ref = oracle_mod.Oracle(1, (6.4, 6.6), 1.0, 0.05, 4, 5)
    for s in (o, ref):
        s.load_positions(np.array([[3.7, 3.8]]))
    same = 0
    for _ in range(400):
        o.sub_sweep(0); ref.sub_sweep(0); o.sub_sweep(1); ref.sub_sweep(1); o.sub_sweep(2); ref.sub_sweep(2); o.sub_sweep(3); ref.sub_sweep(3)
        if ref.acceptance()[2] > 0:
            break
        assert np.array_equal(o.get_positions(), ref.get_positions())
        same += 1
    assert same >= 3 and ref.acceptance()[2] > 0 and o.acceptance()[2] == 0
