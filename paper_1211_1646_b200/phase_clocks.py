"""Per-phase cycle counts of the fused tile kernel (k_tile_sweep), from clock64() marks at its phase boundaries.

    python -m paper_1211_1646_b200.phase_clocks [--workload C3] [--sweeps 200]

Builds an instrumented copy of the library (-DMPMC_PHASE_CLOCKS, its own .so; the shipped library carries no marks),
runs the workload on cuda:0 and prints, over the tiles of the last few sweeps, the mean and the maximum number of SM
cycles each phase took.  The figures quoted in profiles/*ncu_full.md come from this script.
"""
from __future__ import annotations

import argparse
import os

import numpy as np

PHASES = ["wait for the previous sweep", "load tile + halo", "sub-sweep 1", "sub-sweep 2", "sub-sweep 3", "sub-sweep 4",
          "shift + counters"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--sweeps", type=int, default=200)
    ap.add_argument("--samples", type=int, default=20, help="launches whose marks are read")
    ap.add_argument("--dump", default="", help="write the per-tile mean cycles of every phase to this .npy file")
    ap.add_argument("--define", action="append", default=[], help="extra -D for the instrumented build (experiments)")
    ap.add_argument("--burst", type=int, default=10, help="back-to-back sweeps before each read (the last one's marks are read)")
    ap.add_argument("--resident", action="store_true",
                    help="small systems: the cluster-resident kernel's cycle sums (sub-sweeps, barriers, shift) instead of the tile kernel's marks")
    ap.add_argument("--fp32", action="store_true", help="run the workload in fp32 whatever its own precision (with --resident)")
    args = ap.parse_args()
    from . import build
    lib = os.path.join(build.HERE, "libmpmc_b200_phase_clocks.so")
    build.build(extra_flags=["-DMPMC_PHASE_CLOCKS"] + [f"-D{d}" for d in args.define], lib=lib)
    os.environ["MPMC_B200_LIB"] = lib
    import torch
    from . import inputs as I
    from .binding import Mpmc
    w = I.CONFIGS[args.workload]
    xy, box = I.workload_inputs(w)
    if args.resident:
        g = Mpmc(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=w.fp32 or args.fp32, w_target=w.w_target, disc=w.disc)
        cfg = g.config()
        if not cfg["resident_ctas"]:
            raise SystemExit(f"{w.name} does not run on the cluster-resident kernel (too large, or n_s != 4)")
        g.load_positions(torch.as_tensor(xy, device="cuda"))
        g.sweep(args.sweeps)
        g.sweep(args.sweeps)
        pc = g.phase_clocks()
        if pc is None:
            raise SystemExit("this library was built without -DMPMC_PHASE_CLOCKS")
        pc = pc.astype(np.float64)
        per = pc[:, 1:] / pc[:, :1]                  # cycles per sweep
        print(f"{w.name} ({'fp32' if (w.fp32 or args.fp32) else 'fp64'}): cluster of {cfg['resident_ctas']} CTAs ({cfg['resident_cx']} x "
              f"{cfg['resident_cy']} tiles of ~{g.M // cfg['resident_ctas']} cells), {cfg['resident_smem']} B shared memory per CTA; one launch "
              f"of {int(pc[0, 0])} sweeps; SM cycles per sweep, thread 0 of every CTA (mean, max over CTAs):")
        for i, name in enumerate(["four sub-sweeps", "five cluster barriers (incl. waiting for the slowest CTA)", "shift + set-up",
                                  "whole sweep"]):
            print(f"  {name:56s} {per[:, i].mean():9.0f} {per[:, i].max():9.0f}")
        return
    g = Mpmc(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=w.fp32, w_target=w.w_target, disc=w.disc,
             resident=False)                         # the marks are the TILE kernel's: keep small systems on it
    g.load_positions(torch.as_tensor(xy, device="cuda"))
    g.sweep(args.sweeps)
    rows = []
    for _ in range(args.samples):
        g.sweep(args.burst)
        pc = g.phase_clocks()
        if pc is None:
            raise SystemExit("this library was built without -DMPMC_PHASE_CLOCKS")
        rows.append(pc.astype(np.int64))
    pc = np.stack(rows)                              # (samples, tiles, marks)
    extra = pc[:, :, 9:] if pc.shape[2] > 9 else None   # marks inside the sort of the sorted variant (0 if unused)
    pc = pc[:, :, :9]
    d = np.diff(pc[:, :, 1:8], axis=2)               # cycles per phase
    t_ns = (pc[:, :, 8] - pc[:, :, 0])               # mark 8 is the nanosecond timer at the end of the tile's work
    launch_ns = pc[:, :, 8].max(axis=1) - pc[:, :, 0].min(axis=1)
    span_ns = pc[:, :, 0].max(axis=1) - pc[:, :, 0].min(axis=1)
    cfg = g.config()
    print(f"{w.name}: {cfg['ntx']} x {cfg['nty']} tiles, {cfg['tile_threads']} threads, {cfg['tile_smem']} B shared memory; "
          f"{args.samples} launches; tile start times within {span_ns.mean():.0f} ns")
    for i in range(d.shape[2]):
        name = PHASES[i + 1] if i + 1 < len(PHASES) else f"phase {i + 1}"
        print(f"  {name:42s} mean {d[:, :, i].mean():9.0f}   max over tiles (mean over launches) {d[:, :, i].max(axis=1).mean():9.0f} cycles")
    if extra is not None and extra[:, :, 0].min() > 0:
        t_load_end = pc[:, :, 2]
        names = ["row occupancy masks", "simple / general masks + prefix sums"]
        ends = [extra[:, :, i] for i in range(2)]
        print("  inside 'load': the sort ends " + ", ".join(f"{n} {(t_load_end - e).mean():.0f}" for n, e in zip(names, ends))
              + " cycles before the end of the phase")
    if extra is not None and extra.shape[2] >= 7 and extra[:, :, 4].min() > 0:
        t1 = pc[:, :, 1]
        pts = [("first barrier", extra[:, :, 2]), ("count bytes requested, copies issued (warp 0)", extra[:, :, 4]),
               ("count bytes arrived (warp 0)", extra[:, :, 5]), ("row masks of all warps (barrier)", extra[:, :, 0]),
               ("classes + prefix sums", extra[:, :, 1]), ("region arrived, queues written", extra[:, :, 6])]
        print("  inside 'load', cycles after its start: " + "; ".join(f"{n} {(e - t1).mean():.0f}" for n, e in pts))
    if extra is not None and extra.shape[2] >= 10 and extra[:, :, 7].min() > 0:
        e, b, a = extra[:, :, 7], extra[:, :, 8], extra[:, :, 9]
        print(f"  before 'load': kernel entry -> dependency wait {(b - e).mean():.0f} cycles (set-up), in the wait {(a - b).mean():.0f} "
              f"(min over tiles {(a - b).min(axis=1).mean():.0f}), wait -> start of 'load' {(pc[:, :, 1] - a).mean():.0f} (control block)")
    if extra is not None and extra.shape[2] >= 4:
        ncrowd = extra[:, :, 3]
        whole = pc[:, :, 7] - pc[:, :, 1]
        has = ncrowd > 0
        if has.any() and (~has).any():
            print(f"  tiles with a crowded cell in their region: {has.mean() * 100:.1f} % of (launch, tile) pairs; whole tile "
                  f"{whole[has].mean():.0f} cycles against {whole[~has].mean():.0f} without; per phase "
                  + ", ".join(f"{d[:, :, i][has].mean() - d[:, :, i][~has].mean():+.0f}" for i in range(d.shape[2])))
    if args.dump:
        np.save(args.dump, d.mean(axis=0))
    tot = pc[:, :, 7] - pc[:, :, 1]
    print(f"  {'whole tile':42s} mean {tot.mean():9.0f}   max {tot.max(axis=1).mean():9.0f} cycles")
    print(f"  in nanoseconds: a tile takes {t_ns.mean():.0f} (slowest {t_ns.max(axis=1).mean():.0f}); first start to last end of a launch "
          f"{launch_ns.mean():.0f}; the launch period less that is the hand-over between sweeps")


if __name__ == "__main__":
    main()
