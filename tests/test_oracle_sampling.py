"""Statistical pins for the oracle (CPU only): what the paper's detailed-balance argument
and textbook hard-disk results fix, none of it computed by the oracle itself.

  * isolated disk: acceptance -> (1 - d/(2 wx)) (1 - d/(2 wy))            (closed form)
  * N = 2 on a small torus: relative vector uniform on the torus minus a disc of radius sigma,
    absolute position uniform                                               (closed form per bin, chi^2)
  * N = 3: pair-distance law against direct sampling (uniform placement, reject on overlap)
  * N = 64: pair-distance histogram against an independently written serial MC (Fig. 1)
  * low-density pressure against the hard-disk virial series
  * contact histogram against brute-force numpy pair distances; the fit on the paper's model n(r) (L382)
All seeds are fixed, so every test is deterministic; thresholds were chosen once with margin.
"""
import math

import numpy as np
import pytest
from scipy import stats

from paper_1211_1646_b200 import inputs as I
from tests.helpers import serial


@pytest.mark.parametrize("fp32", [False, True])
@pytest.mark.parametrize("d,box", [(0.5, (2.6, 2.6)), (0.08, (2.2, 2.8))])
def test_isolated_disk_acceptance(oracle_mod, fp32, d, box):
    o = oracle_mod.Oracle(1, box, 1.0, d, 4, 11, fp32=fp32)
    o.load_positions(np.array([[0.3, 0.4]]))
    o.sweep(30000)
    att, acc, rej_b, rej_o = o.acceptance()
    assert att == 4 * 30000 and rej_o == 0
    expect = (1 - d / (2 * o.wx)) * (1 - d / (2 * o.wy))
    assert acc / att == pytest.approx(expect, abs=0.006)


@pytest.mark.parametrize("fp32", [False, True])
@pytest.mark.parametrize("d,box", [(0.5, (2.6, 2.6)), (0.3, (2.2, 2.8))])
def test_isolated_disk_acceptance_disc_proposal(oracle_mod, fp32, d, box):
    """The paper's proposal, uniform in the disc of radius d (L190).  For a position uniform in the cell the move stays
    with probability 1 - E|dx|/wx - E|dy|/wy + E|dx dy|/(wx wy), E|dx| = 4d/(3 pi), E|dx dy| = d^2/(2 pi) (disc
    integrals, worked out by hand) — different from the square proposal's (1 - d/2wx)(1 - d/2wy)."""
    o = oracle_mod.Oracle(1, box, 1.0, d, 4, 13, fp32=fp32, disc=True)
    o.load_positions(np.array([[0.3, 0.4]]))
    o.sweep(30000)
    att, acc, rej_b, rej_o = o.acceptance()
    assert att == 4 * 30000 and rej_o == 0
    expect = 1 - 4 * d / (3 * math.pi) * (1 / o.wx + 1 / o.wy) + d * d / (2 * math.pi * o.wx * o.wy)
    square = (1 - d / (2 * o.wx)) * (1 - d / (2 * o.wy))
    assert acc / att == pytest.approx(expect, abs=0.006)
    assert abs(acc / att - square) > 0.02            # the two proposals are told apart


def test_disc_proposal_displacements_are_uniform_in_the_disc(oracle_mod):
    """One disk in a wide cell (boundary rejections rare), n_s = 1: the displacement of every accepted move is a position
    difference.  |delta| <= d always; r^2/d^2 uniform on [0, 1] (chi^2), mean r^2 = d^2/2 (the square would give 2d^2/3);
    the angle uniform (chi^2 over 8 sectors)."""
    d = 0.7
    o = oracle_mod.Oracle(1, (60.0, 60.0), 1.0, d, 1, 5, fp32=False, w_target=30.0, disc=True)
    assert (o.mx, o.my) == (2, 2)
    o.load_positions(np.array([[15.0, 15.0]]))
    prev = o.get_positions()[0].copy()
    disp = []
    for _ in range(6000):
        o.sweep(1)
        cur = o.get_positions()[0]
        dd = cur - prev
        dd -= np.round(dd / 60.0) * 60.0
        if np.abs(dd).max() > 0:
            disp.append(dd)
        prev = cur.copy()
    disp = np.array(disp)
    assert len(disp) > 5000
    r2 = (disp ** 2).sum(axis=1) / d ** 2
    assert r2.max() <= 1.0 + 1e-12
    assert r2.mean() == pytest.approx(0.5, abs=0.02)
    assert stats.chisquare(np.histogram(r2, bins=10, range=(0, 1))[0]).pvalue > 1e-3
    ang = np.arctan2(disp[:, 1], disp[:, 0])
    assert stats.chisquare(np.histogram(ang, bins=8, range=(-math.pi, math.pi))[0]).pvalue > 1e-3


def _excluded_disc_law(K, Le, sub=80):
    xs = (np.arange(K * sub) + 0.5) / (K * sub) * Le[0] - Le[0] / 2
    ys = (np.arange(K * sub) + 0.5) / (K * sub) * Le[1] - Le[1] / 2
    X, Y = np.meshgrid(xs, ys, indexing="ij")
    ok = (X * X + Y * Y) >= 1.0
    return ok.reshape(K, sub, K, sub).sum(axis=(1, 3)) / ok.sum()


@pytest.mark.parametrize("fp32,seed,disc", [(False, 1, False), (True, 2, False), (False, 3, True)])
def test_two_disks_sample_uniform_law(oracle_mod, fp32, seed, disc):
    L = (2.6, 2.9)
    o = oracle_mod.Oracle(2, L, 1.0, 0.4, 4, seed, fp32=fp32, disc=disc)
    assert (o.mx, o.my) == (2, 2)          # one neighbour cell appears at two image offsets (A11)
    o.load_positions(np.array([[0.5, 0.5], [1.8, 1.9]]))
    S = 20000
    rel = np.zeros((S, 2))
    p0 = np.zeros((S, 2))
    for i in range(S):
        o.sweep(10)
        p = o.get_positions()
        p0[i] = p[0]
        rel[i] = p[1] - p[0]
    Le = np.array(o.L_eff)
    rel -= Le * np.round(rel / Le)
    assert np.all((rel ** 2).sum(axis=1) >= 1.0 - 1e-5)
    K = 12
    ex = _excluded_disc_law(K, Le)
    h, _, _ = np.histogram2d(rel[:, 0], rel[:, 1], bins=K, range=[[-Le[0] / 2, Le[0] / 2], [-Le[1] / 2, Le[1] / 2]])
    assert h[ex == 0].sum() == 0
    m = ex > 5 / S
    chi = ((h[m] - S * ex[m]) ** 2 / (S * ex[m])).sum()
    assert stats.chi2.sf(chi, m.sum() - 1) > 1e-3
    h0, _, _ = np.histogram2d(p0[:, 0], p0[:, 1], bins=8, range=[[0, Le[0]], [0, Le[1]]])
    assert stats.chisquare(h0.ravel()).pvalue > 1e-3


def test_three_disks_match_direct_sampling(oracle_mod):
    L = (4.3, 4.5)
    o = oracle_mod.Oracle(3, L, 1.0, 0.5, 4, 3)
    assert (o.mx, o.my) == (4, 4)
    o.load_positions(np.array([[0.5, 0.5], [2.0, 2.0], [3.5, 0.9]]))
    Le = np.array(o.L_eff)
    S = 15000

    def pair_d(p):
        out = []
        for a, b in ((0, 1), (0, 2), (1, 2)):
            dlt = p[a] - p[b]
            dlt -= Le * np.round(dlt / Le)
            out.append(math.hypot(*dlt))
        return out

    mc = np.zeros((S, 3))
    for i in range(S):
        o.sweep(8)
        mc[i] = pair_d(o.get_positions())
    rng = np.random.default_rng(99)
    direct = []
    while len(direct) < S:
        p = rng.uniform(0, 1, size=(3, 2)) * Le
        dd = pair_d(p)
        if min(dd) >= 1.0:
            direct.append(dd)
    direct = np.array(direct)
    assert mc.min() >= 1.0 - 1e-12
    # smallest pair distance and the all-pairs law, two-sample tests
    assert stats.ks_2samp(mc.min(axis=1), direct.min(axis=1)).pvalue > 1e-3
    edges = np.linspace(1.0, 0.5 * math.hypot(*Le), 16)
    h1, _ = np.histogram(mc.ravel(), bins=edges)
    h2, _ = np.histogram(direct.ravel(), bins=edges)
    assert stats.chi2_contingency(np.array([h1, h2]))[1] > 1e-3


def _gr_from_positions(p, Le, sigma, rmax, nbins):
    d = p[:, None, :] - p[None, :, :]
    d -= Le * np.round(d / Le)
    r = np.sqrt((d ** 2).sum(-1))[np.triu_indices(len(p), 1)]
    b = np.floor((r - sigma) / ((rmax - sigma) / nbins)).astype(int)
    b = b[(b >= 0) & (b < nbins)]
    return np.bincount(b, minlength=nbins).astype(float)


def test_agrees_with_serial_mc(oracle_mod):
    n_side, phi = 8, 0.40
    xy, box = I.jittered_lattice(n_side, phi, seed=5)
    N = n_side * n_side
    o = oracle_mod.Oracle(N, box, 1.0, 0.3, 4, 21)
    o.load_positions(xy)
    Le = np.array(o.L_eff)
    rmax, nbins, S = 2.0, 20, 3000
    o.sweep(500)
    h_mpmc = np.zeros((S, nbins))
    for i in range(S):
        o.sweep(4)
        h_mpmc[i] = _gr_from_positions(o.get_positions(), Le, 1.0, rmax, nbins)
    h_ser, acc = serial.pair_histograms(xy, tuple(Le), 1.0, 0.3, 77, 500, S, 4, rmax, nbins)
    assert 0.2 < acc < 0.9

    def mean_err(h, nblock=30):
        blocks = h[: (len(h) // nblock) * nblock].reshape(nblock, -1, h.shape[1]).mean(axis=1)
        return h.mean(axis=0), blocks.std(axis=0, ddof=1) / math.sqrt(nblock)

    m1, e1 = mean_err(h_mpmc)
    m2, e2 = mean_err(h_ser)
    z = (m1 - m2) / np.sqrt(e1 ** 2 + e2 ** 2)
    assert np.abs(z).max() < 4.5, z
    assert (z ** 2).sum() < stats.chi2.isf(1e-3, nbins)
    # the two curves are the same to about a percent where the counts are large
    assert np.abs(m1 / m2 - 1).max() < 0.05


def test_contact_histogram_matches_brute_force(oracle_mod):
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    for fp32 in (False, True):
        o = oracle_mod.Oracle(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=fp32)
        o.load_positions(xy)
        o.sweep(20)
        for dr, nbins in ((0.005, 20), (0.01, 60), (1e-3, 20)):
            h = o.contact_histogram(dr, nbins)
            p = o.get_positions()
            Le = np.array(o.L_eff)
            from scipy.spatial import cKDTree
            tree = cKDTree(np.minimum(p, np.nextafter(Le, 0)), boxsize=Le)
            pairs = tree.query_pairs(w.sigma + dr * nbins + 1e-9, output_type="ndarray")
            dlt = p[pairs[:, 0]] - p[pairs[:, 1]]
            dlt -= Le * np.round(dlt / Le)
            r = np.sqrt((dlt ** 2).sum(1))
            b = np.floor((r - w.sigma) / dr).astype(int)
            ref = np.bincount(b[(b >= 0) & (b < nbins)], minlength=nbins)
            assert h.sum() > 50
            # identical up to pairs whose distance sits within rounding of a bin edge
            assert np.abs(h.astype(np.int64) - ref).sum() <= (6 if fp32 else 2)


def test_fit_unbiased_on_paper_model_distribution(oracle_mod):
    # n(r) = 30 exp(-30 r), dr = 1e-4 sigma, c = 0.02 sigma, degree 5 -> bias < 1e-5
    sigma, dr, c, degree = 1.0, 1e-4, 0.02, 5
    nb = int(round(c / dr))
    r_lo = dr * np.arange(nb)
    r_hi = dr * np.arange(1, nb + 1)
    n_bin = np.exp(-30 * r_lo) - np.exp(-30 * r_hi)          # exact bin integrals of 30 e^{-30 r}
    R_lo, R_hi = sigma + r_lo, sigma + r_hi
    R = (2 / 3) * (R_hi ** 3 - R_lo ** 3) / (R_hi ** 2 - R_lo ** 2)     # eq. 6
    est = oracle_mod.fit_contact(R, n_bin / dr, sigma, degree)
    assert abs(est / 30.0 - 1.0) < 1e-5
    # a mis-centred sample point (bin edge instead of eq. 6) is far outside that bound
    assert abs(oracle_mod.fit_contact(R_lo, n_bin / dr, sigma, degree) / 30.0 - 1.0) > 1e-4


def test_g_of_r_normalisation_ideal_gas(oracle_mod):
    # uncorrelated points: expected unordered pairs in a thin annulus = N (N-1)/2 * 2 pi r dr / A, so g -> 1
    N, Le, sigma, dr, nb = 4000, (50.0, 40.0), 1.0, 0.01, 10
    R, g, rho = oracle_mod.g_of_r(np.full(nb, 1.0), N, Le, sigma, dr)
    assert rho == pytest.approx(2.0)
    r_mid = sigma + dr * (np.arange(nb) + 0.5)
    expected_pairs = 0.5 * N * (N - 1) * 2 * math.pi * r_mid * dr / (Le[0] * Le[1])
    R2, g2, _ = oracle_mod.g_of_r(expected_pairs, N, Le, sigma, dr)
    assert np.allclose(g2, 1.0, atol=2e-3)
    assert np.all((R2 > sigma + dr * np.arange(nb)) & (R2 < sigma + dr * np.arange(1, nb + 1)))


VIRIAL = (1.0, 2.0, 3.1280, 4.2579, 5.337, 6.363)   # Z = sum_k c_k phi^k (B3, B4 exact)


@pytest.mark.parametrize("phi,fp32", [(0.05, False), (0.10, True), (0.20, False)])
def test_low_density_pressure_matches_virial_series(oracle_mod, phi, fp32):
    n_side = 16
    N = n_side * n_side
    xy, box = I.jittered_lattice(n_side, phi, seed=3)
    o = oracle_mod.Oracle(N, box, 1.0, 0.5, 4, 17, fp32=fp32)
    o.load_positions(xy)
    o.sweep(400)
    dr, nbins, degree = 0.01, 20, 2
    H = np.zeros(nbins)
    S = 4000
    for _ in range(S):
        o.sweep(3)
        H += o.contact_histogram(dr, nbins)
    g0, p_star = oracle_mod.pressure_from_histogram(H / S, N, o.L_eff, 1.0, dr, degree)
    rho = N / (o.L_eff[0] * o.L_eff[1])
    Z = p_star / rho                                    # P sigma^2/kT / (rho sigma^2)
    phi_eff = rho * math.pi / 4                         # the simulated box is L_eff (fp32: differs by ~1e-8)
    assert Z == pytest.approx(1 + 2 * phi_eff * g0, rel=1e-12)   # eq. 4 rewritten with phi = rho pi sigma^2/4
    Z_virial = sum(c * phi ** k for k, c in enumerate(VIRIAL))
    assert Z == pytest.approx(Z_virial, rel=0.006)
