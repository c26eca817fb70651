"""Seeded synthetic input generators (shared by the oracle tests, the GPU tests and bench.py).

This module holds NONE of the method's arithmetic (no cell list, no Philox, no trial moves):
it only lays disks on a jittered triangular lattice.  Both the oracle and the CUDA path take the
arrays produced here as plain inputs.

Recipe (BASELINE.json `configs`, reading A14):
  * n x n triangular lattice, site (i, j) at ((i + (j mod 2)/2) a, j a sqrt(3)/2),
    a = sigma sqrt(pi / (2 sqrt(3) phi)), periodic box (n a, n a sqrt(3)/2)  -> aspect 2/sqrt(3);
    phi = rho pi (sigma/2)^2 is the paper's packing fraction.
  * every disk is displaced by an independent per-coordinate U[-jit, +jit] offset (jit = 0.05 sigma);
    while any pair of lattice neighbours overlaps (centre distance < sigma), the higher-index disk of
    each overlapping pair redraws its offset.  Lattice sites start at x = a/4, y = a sqrt(3)/4 so no
    disk sits on the box edge.
These stand in for the paper's equilibrated configurations, which do not exist here.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config: everything `mpmc_create` needs plus the run length."""
    name: str
    n_side: int          # lattice is n_side x n_side
    phi: float
    sigma: float
    d: float             # maximum displacement (per coordinate), in units of length
    n_s: int             # trial moves per active cell per sub-sweep (the paper's n_M)
    sweeps: int
    seed: int
    fp32: bool
    jitter: float = 0.05
    w_target: float = 0.0   # requested minimum cell width (0: smallest width >= sigma that divides the box)
    disc: bool = False      # trial displacement uniform in the disc of radius d instead of the square
    melt: int = 0           # "melted for `melt` serial-equivalent sweeps" (BASELINE C5, reading A15): the caller runs the
                            # method with preparation seed 999 until attempted >= melt * N before the measured run

    @property
    def N(self) -> int:
        return self.n_side * self.n_side


# BASELINE.json `configs`, in order.  C2 runs in both precisions (fp64 listed; tests also use fp32).
CONFIGS = {
    "C1": Workload("C1", 64, 0.50, 1.0, 0.25, 4, 100, 1, fp32=False),
    "C2": Workload("C2", 256, 0.70, 1.0, 0.10, 4, 1000, 1, fp32=False),
    "C3": Workload("C3", 1024, 0.716, 1.0, 0.08, 4, 1000, 1, fp32=True),
    "C4": Workload("C4", 4096, 0.720, 1.0, 0.06, 8, 200, 1, fp32=True),
    "C5": Workload("C5", 1024, 0.30, 1.0, 0.5, 4, 1000, 1, fp32=True, melt=100),
}

# The paper's own regime as a second workload: cell width just under sqrt(2) sigma (L152), disc-shaped
# displacement of radius d = 0.16 sigma and n_M = 4 (L190, L358), phi = 0.698, single precision (L390), sizes next to
# Table 4's N = 253^2 ... 3040^2 (L411).  Same jittered triangular lattice in the 2/sqrt(3) box (the paper's box is square).
for _n in (256, 768, 1536, 3072):
    CONFIGS[f"P{_n}"] = Workload(f"P{_n}", _n, 0.698, 1.0, 0.16, 4, 100, 1, fp32=True, w_target=1.40, disc=True)


def lattice_constant(phi: float, sigma: float = 1.0) -> float:
    return sigma * math.sqrt(math.pi / (2.0 * math.sqrt(3.0) * phi))


def box_for(n_side: int, phi: float, sigma: float = 1.0) -> tuple[float, float]:
    a = lattice_constant(phi, sigma)
    return n_side * a, n_side * a * math.sqrt(3.0) / 2.0


def _neighbour_overlaps(x: np.ndarray, y: np.ndarray, Lx: float, Ly: float, sigma: float) -> np.ndarray:
    """Boolean (n, n) mask: disk [j, i] overlaps a lattice neighbour of LOWER linear index j*n+i.

    x, y are (n, n) arrays indexed [j, i].  The six triangular-lattice neighbours of (i, j) are
    (i±1, j) and, in rows j±1, columns i and i+1 (j odd) or i-1 and i (j even).
    """
    n = x.shape[0]
    jj, ii = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    lin = jj * n + ii
    bad = np.zeros((n, n), dtype=bool)
    odd = (jj % 2) == 1
    s2 = sigma * sigma

    def check(nj, ni):
        nj = nj % n
        ni = ni % n
        dx = x[nj, ni] - x
        dy = y[nj, ni] - y
        dx -= Lx * np.round(dx / Lx)
        dy -= Ly * np.round(dy / Ly)
        ov = (dx * dx + dy * dy) < s2
        return ov & (lin[nj, ni] < lin)

    bad |= check(jj, ii - 1)
    bad |= check(jj, ii + 1)
    for dj in (-1, 1):
        c0 = np.where(odd, ii, ii - 1)
        bad |= check(jj + dj, c0)
        bad |= check(jj + dj, c0 + 1)
    return bad


def jittered_lattice(n_side: int, phi: float, sigma: float = 1.0, jitter: float = 0.05,
                     seed: int = 1) -> tuple[np.ndarray, tuple[float, float]]:
    """Return (xy, (Lx, Ly)): xy is (N, 2) float64, disk index = j*n_side + i, all inside [0, L)."""
    n = int(n_side)
    a = lattice_constant(phi, sigma)
    Lx, Ly = box_for(n, phi, sigma)
    if a <= sigma or n % 2:
        raise ValueError("need an even n_side and a lattice constant above sigma")
    rng = np.random.Generator(np.random.Philox(key=int(seed)))
    jj, ii = np.meshgrid(np.arange(n, dtype=np.float64), np.arange(n, dtype=np.float64), indexing="ij")
    x0 = (ii + 0.5 * (jj % 2) + 0.25) * a
    y0 = (jj + 0.5) * (a * math.sqrt(3.0) / 2.0)
    jit = jitter * sigma
    ox = rng.uniform(-jit, jit, size=(n, n))
    oy = rng.uniform(-jit, jit, size=(n, n))
    for _ in range(1000):
        bad = _neighbour_overlaps(x0 + ox, y0 + oy, Lx, Ly, sigma)
        nbad = int(bad.sum())
        if nbad == 0:
            break
        ox[bad] = rng.uniform(-jit, jit, size=nbad)
        oy[bad] = rng.uniform(-jit, jit, size=nbad)
    else:  # pragma: no cover
        raise RuntimeError("jitter rejection did not converge")
    xy = np.stack([(x0 + ox).ravel(), (y0 + oy).ravel()], axis=1)
    xy[:, 0] %= Lx
    xy[:, 1] %= Ly
    return np.ascontiguousarray(xy), (Lx, Ly)


def workload_inputs(w: Workload) -> tuple[np.ndarray, tuple[float, float]]:
    return jittered_lattice(w.n_side, w.phi, w.sigma, w.jitter, w.seed)


def random_dilute(N: int, L: tuple[float, float], sigma: float, seed: int) -> np.ndarray:
    """N disks placed uniformly at random without overlap (random sequential addition); tiny/dilute
    test systems only (O(N^2))."""
    rng = np.random.Generator(np.random.Philox(key=int(seed)))
    pts: list[tuple[float, float]] = []
    Lx, Ly = L
    tries = 0
    while len(pts) < N:
        tries += 1
        if tries > 100000 * N:
            raise RuntimeError("random placement failed")
        px, py = rng.uniform(0, Lx), rng.uniform(0, Ly)
        ok = True
        for qx, qy in pts:
            dx = px - qx
            dy = py - qy
            dx -= Lx * round(dx / Lx)
            dy -= Ly * round(dy / Ly)
            if dx * dx + dy * dy < sigma * sigma * 1.0001:
                ok = False
                break
        if ok:
            pts.append((px, py))
    return np.asarray(pts, dtype=np.float64).reshape(N, 2)

# Small systems ("launch overhead" below N ~ 1e5): C3's parameters at N = 32^2 and 64^2, and
# the paper's regime at N = 64^2 and 128^2 — sizes at which the state lives in one thread-block cluster's shared memory
# (csrc/cluster.cuh).  bench.py --workload S64 [--no-resident] times both mappings.
for _n in (32, 64):
    CONFIGS[f"S{_n}"] = Workload(f"S{_n}", _n, 0.716, 1.0, 0.08, 4, 1000, 1, fp32=True)
for _n in (64, 128):
    CONFIGS[f"P{_n}"] = Workload(f"P{_n}", _n, 0.698, 1.0, 0.16, 4, 1000, 1, fp32=True, w_target=1.40, disc=True)

