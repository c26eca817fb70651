#!/usr/bin/env python
"""One equation-of-state point with the paper's pressure estimator (eq. 4-6): pair-distance histogram
near contact with dr = 1e-4 sigma on (sigma, 1.02 sigma], sampled every 200 sweeps, degree-5 polynomial fit extrapolated to
r = sigma.  Default: N = 256^2, phi = 0.698, the liquid point of Table 2 (L399: P* = 9.1709(1) MPMC, 9.1708(4) event-chain).
Uses the CUDA library only (needs a GPU).  The box is the 2/sqrt(3) rectangle of the BASELINE configs, not the paper's
square, and the proposal is the square of reading A2; neither changes the ensemble.

  python -m paper_1211_1646_b200.eos_check [--n 256] [--phi 0.698] [--equil 400000] [--sweeps 2000000] [--d 0.12]
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=256, help="lattice side: N = n^2 disks")
    ap.add_argument("--phi", type=float, default=0.698)
    ap.add_argument("--d", type=float, default=0.12, help="maximum displacement per coordinate, in sigma")
    ap.add_argument("--n-s", type=int, default=4)
    ap.add_argument("--equil", type=int, default=400_000, help="sweeps discarded before sampling")
    ap.add_argument("--sweeps", type=int, default=2_000_000, help="sampled sweeps")
    ap.add_argument("--every", type=int, default=200, help="sweeps between histogram samples (L384)")
    ap.add_argument("--blocks", type=int, default=10, help="blocks for the error estimate")
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--fp64", action="store_true")
    ap.add_argument("--w-target", type=float, default=0.0, help="minimum cell width (1.40: the paper's regime, L152)")
    ap.add_argument("--disc", action="store_true", help="disc-shaped displacement (the paper's, L190)")
    ap.add_argument("--no-particle-shuffle", action="store_true", help="ablation of Table 1 (L134-142)")
    ap.add_argument("--no-set-shuffle", action="store_true", help="ablation of Table 1 (L134-142)")
    args = ap.parse_args()

    import torch
    from . import inputs as I
    from .binding import Mpmc
    xy, box = I.jittered_lattice(args.n, args.phi, seed=args.seed)
    N = args.n * args.n
    sim = Mpmc(N, box, 1.0, args.d, args.n_s, args.seed, fp32=not args.fp64, device="cuda:0", w_target=args.w_target,
               disc=args.disc, particle_shuffle=not args.no_particle_shuffle, set_shuffle=not args.no_set_shuffle)
    sim.load_positions(torch.as_tensor(xy, device="cuda:0"))
    dr, nbins, degree = 1e-4, 200, 5                      # L382
    t0 = time.time()
    sim.sweep(args.equil)
    torch.cuda.synchronize()
    t_eq = time.time() - t0
    a0 = sim.acceptance()
    nsamp = args.sweeps // args.every
    per_block = max(1, nsamp // args.blocks)
    # the estimator (eq. 4-6, degree-5 fit) lives behind the C ABI: mpmc_pressure_accumulate adds a sample on the device
    # without a host synchronisation, mpmc_pressure_accumulated fits a block, mpmc_pressure_from_histogram the whole run
    hist_all = np.zeros(nbins, dtype=np.uint64)
    p_blocks = []
    t0 = time.time()
    for _ in range(args.blocks):
        sim.pressure_reset()
        for _ in range(per_block):
            sim.sweep(args.every)
            sim.pressure_accumulate(dr, nbins)
        h, n, _, p_b = sim.pressure_accumulated(degree, nbins)
        assert n == per_block
        hist_all += h
        p_blocks.append(p_b)
    torch.cuda.synchronize()
    t_run = time.time() - t0
    a1 = sim.acceptance()
    L = sim.L_eff
    g_all, p_all = sim.pressure_from_histogram(hist_all, per_block * args.blocks, dr, degree)
    p_blocks = np.array(p_blocks)
    out = {
        "N": N, "phi": args.phi, "box": list(L), "cells": [sim.mx, sim.my], "d": args.d, "n_s": args.n_s,
        "dtype": "f64" if args.fp64 else "f32", "w_target": args.w_target, "disc": args.disc,
        "particle_shuffle": not args.no_particle_shuffle, "set_shuffle": not args.no_set_shuffle, "equil_sweeps": args.equil, "sampled_sweeps": per_block * args.blocks * args.every,
        "samples": per_block * args.blocks, "P_star": p_all, "g_contact": g_all,
        "P_star_block_mean": float(p_blocks.mean()), "P_star_stderr": float(p_blocks.std(ddof=1) / np.sqrt(args.blocks)),
        "P_star_blocks": [float(v) for v in p_blocks],
        "acceptance": (a1[1] - a0[1]) / max(1, a1[0] - a0[0]),
        "paper": {"P_star_MPMC": 9.1709, "P_star_event_chain": 9.1708, "citation": "PAPER.md L399 (Table 2, phi = 0.698, N = 256^2)"}
        if abs(args.phi - 0.698) < 1e-9 else None,
        "moves_per_s_incl_sampling": (a1[0] - a0[0]) / t_run, "seconds": {"equilibration": t_eq, "sampling": t_run},
        "path_sweeps": sim.path_sweeps(),
    }
    print(json.dumps(out))


if __name__ == "__main__":
    main()
