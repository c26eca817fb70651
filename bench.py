#!/usr/bin/env python
"""bench.py — hard-disk trial moves/s of the checkerboard cell sweep (BASELINE.json metric) on B200.

One "step" = one pass of the whole hot path over one batch of synthetic input:
  cell-list build from N x 2 doubles  ->  S sweeps (four sub-sweeps + shift each; one fused tile-kernel launch per
  sweep)  ->  contact histogram  ->  unpack  ->  read the move counters.
`value`  : inputs resident in HBM when the timed region starts (CUDA events on the library's stream).
`e2e`    : the same step through the same C-ABI calls with HOST buffers: pinned host -> device copy of the
           positions and device -> host copy of the result inside the timed region.
Trial moves are taken from the exact device counters (attempted = n_s per non-empty active cell).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C3] [--sweeps S]
N > 1: launched by torch.distributed.run, one rank per GPU, independent replicas (DESIGN.md "Multi-GPU:
replicas only" — the paper runs one GPU, L390); value = all ranks' moves / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1211_1646_b200 import inputs as I  # noqa: E402

METRIC = "hard-disk trial moves/sec"
UNIT = "trial moves/s"


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for nm, v in zip(names, r[4:8]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def algorithmic_bytes_per_sweep(N: int, M: int, fp32: bool) -> float:
    """each of the four sub-sweeps reads every cell once (e bytes per disk + 1 count byte per cell)
    and writes back the active quarter, the shift reads and writes everything: 7 (e N + M) per sweep."""
    e = 8 if fp32 else 16
    return 7.0 * (e * N + M)          # 4 x 1.25 passes + shift read + shift write


def fused_floor_bytes_per_sweep(N: int, M: int, fp32: bool) -> float:
    """What a sweep fused into one pass (the tile kernel) must move: read everything once, write everything once."""
    e = 8 if fp32 else 16
    return 2.0 * (e * N + M)


def aggregate(dist, dev, ms_and_moves):
    """Whole-job figures of N independent replicas: MAX over ranks of the device times, SUM over ranks of the moves.
    ms_and_moves = [ms, ms_e2e, moves, moves_e2e]; returns the same four, reduced (unchanged without dist)."""
    if dist is None:
        return list(ms_and_moves)
    import torch
    t = torch.tensor(ms_and_moves[:2], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    m = torch.tensor(ms_and_moves[2:], dtype=torch.float64, device=dev)
    dist.all_reduce(m, op=dist.ReduceOp.SUM)
    return t.tolist() + m.tolist()


def oracle_inputs(O, w):
    """The workload's input for the CPU legs: no oracle input ever comes from the CUDA path, so a workload that starts
    from a melted lattice (reading A15) is melted here by the oracle itself."""
    xy, box = I.workload_inputs(w)
    if w.melt:
        prep = O.Oracle(w.N, box, w.sigma, w.d, w.n_s, 999, fp32=w.fp32, w_target=w.w_target, disc=w.disc)
        prep.load_positions(xy)
        while prep.acceptance()[0] < w.melt * w.N:
            prep.sweep(10)
        xy = prep.get_positions()
    return xy, box


def run_reference(args, w):
    """--impl reference: the oracle as it stands, single thread, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    O.build()
    xy, box = oracle_inputs(O, w)
    o = O.Oracle(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=w.fp32, w_target=w.w_target, disc=w.disc)
    o.load_positions(xy)
    sample_sweeps = max(1, args.ref_sweeps)
    for _ in range(args.warmup):
        o.sweep(1)
    a0 = o.acceptance()[0]
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.sweep(sample_sweeps)
    dt = time.perf_counter() - t0
    moves = o.acceptance()[0] - a0
    val = moves / dt
    sample = f"{args.steps} steps x {sample_sweeps} sweeps of {w.name} (N={w.N}), after {args.warmup} warm-up sweeps"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32" if w.fp32 else "f64",
        "data": "synthetic", "config": workload_config(w, sample_sweeps),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def workload_config(w, sweeps):
    return {"workload": f"{w.name}: N={w.N} hard disks ({w.n_side}x{w.n_side} jittered triangular lattice), "
                        f"phi={w.phi}, d={w.d} sigma, n_s={w.n_s}, {'fp32' if w.fp32 else 'fp64'} positions"
                        + (f", cell width >= {w.w_target} sigma" if w.w_target else "")
                        + (", disc-shaped displacement" if w.disc else ""),
            "sweeps_per_step": sweeps, "seed": w.seed}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=11, help="timed steps (11: the paper's protocol, median of 11 runs, PAPER.md L421)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3", choices=sorted(I.CONFIGS))
    ap.add_argument("--sweeps", type=int, default=0, help="sweeps per step (0: the workload's own count; C3: 1,000)")
    ap.add_argument("--ref-sweeps", type=int, default=2, help="oracle sweeps per step for --impl reference")
    ap.add_argument("--cpu-baseline-sweeps", type=int, default=15)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-resident", action="store_true",
                    help="small systems on the fused tile kernels instead of the cluster-resident kernel (MPMC_NO_RESIDENT): A/B")
    args = ap.parse_args()
    w = I.CONFIGS[args.workload]
    if args.impl == "reference":
        return run_reference(args, w)

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    from paper_1211_1646_b200 import build
    from paper_1211_1646_b200.binding import Mpmc
    build.build()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=dev)

    S = args.sweeps if args.sweeps > 0 else w.sweeps
    xy_np, box = I.workload_inputs(w)
    if w.melt:                                     # reading A15: the product melts the lattice (preparation seed 999)
        prep = Mpmc(w.N, box, w.sigma, w.d, w.n_s, 999, fp32=w.fp32, device=dev, w_target=w.w_target, disc=w.disc)
        prep.load_positions(torch.from_numpy(xy_np).to(dev))
        while prep.acceptance()[0] < w.melt * w.N:
            prep.sweep(10)
        xy_np = prep.get_positions().cpu().numpy()
        prep.close()
    xy_pinned = torch.from_numpy(xy_np).pin_memory()
    xy_dev = xy_pinned.to(dev)
    out_dev = torch.empty_like(xy_dev)
    out_pinned = torch.empty_like(xy_pinned).pin_memory()
    sim = Mpmc(w.N, box, w.sigma, w.d, w.n_s, w.seed + rank, fp32=w.fp32, device=dev, w_target=w.w_target, disc=w.disc,
               resident=not args.no_resident)   # replicas: seed per rank
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def step_resident():
        sim.load_positions(xy_dev)                    # a3
        sim.sweep(S)                                  # a0-a2
        hist = sim.contact_histogram(0.005, 20)       # a4
        sim.get_positions(out_dev)                    # a5
        return sim.acceptance()[0], hist              # counters (synchronises)

    def step_e2e():
        xy_dev.copy_(xy_pinned, non_blocking=True)    # host -> device inside the timed region
        sim.load_positions(xy_dev)
        sim.sweep(S)
        hist = sim.contact_histogram(0.005, 20)
        sim.get_positions(out_dev)
        out_pinned.copy_(out_dev, non_blocking=True)  # device -> host
        return sim.acceptance()[0], hist

    def timed(fn, K, sampler=None):
        """K timed steps; returns (sum of the step times in ms, sum of the trial moves, per-step rates in moves/s)."""
        total_ms, moves, rates = 0.0, 0, []
        for _ in range(K):
            flush.fill_(1)                            # L2 flush between timed iterations (not timed)
            torch.cuda.synchronize(dev)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            att, _ = fn()
            e1.record()
            torch.cuda.synchronize(dev)
            ms_step = e0.elapsed_time(e1)
            total_ms += ms_step
            moves += att
            rates.append(att / (ms_step * 1e-3))
        return total_ms, moves, rates

    def spread(rates):
        """median with min / max over the timed steps (the paper reports the median of 11 runs)"""
        return {"median": float(np.median(rates)), "min": float(np.min(rates)), "max": float(np.max(rates)), "steps": len(rates)}

    # everything below is enqueued on the library's own stream, so torch.cuda.Event times that stream
    torch.cuda.synchronize(dev)
    torch.cuda.set_stream(sim.stream)
    for _ in range(args.warmup):
        step_resident()
    if dist:
        dist.barrier()
    torch.cuda.synchronize(dev)
    sampler = ClockSampler(local)
    sampler.start()
    ms, moves, rates = timed(step_resident, args.steps)
    clocks = sampler.stop()
    torch.cuda.synchronize(dev)
    if dist:
        dist.barrier()
    for _ in range(max(1, args.warmup // 3)):
        step_e2e()
    ms_e2e, moves_e2e, rates_e2e = timed(step_e2e, args.steps)

    # ---- roofline of the dominant kernel: k_tile_sweep, one launch = one whole sweep (four sub-sweeps + shift),
    #      timed live with CUDA events on the library's stream over S back-to-back launches ----
    sim.load_positions(xy_dev)
    sim.sweep(100)
    a0 = sim.acceptance()[0]
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); sim.sweep(S); e1.record(); torch.cuda.synchronize(dev)
    sweep_ms = e0.elapsed_time(e1) / S
    moves_per_sweep = (sim.acceptance()[0] - a0) / S
    tile_sweeps, general_sweeps = sim.path_sweeps()
    cfg = sim.config()
    e = 8 if w.fp32 else 16
    state_bytes = sim.M * (2 * e + 8 + 1)              # slot pair 0 + its ids + count of every cell, one buffer
    l2_bytes = torch.cuda.get_device_properties(dev).L2_cache_size
    tile_name = "k_tile4_sweep" if (w.disc or w.w_target >= 1.15) else "k_tile_sweep"     # 4-slot / 2-slot tile kernel
    kernel = tile_name if tile_sweeps >= general_sweeps else "k_sweeps"
    resident = cfg["resident_ctas"] > 0                # small system: ONE launch of one cluster runs all S sweeps (cluster.cuh)
    if resident:
        kernel = "k_cluster_sweeps"
    peak, peak_src = peaks()
    alg = algorithmic_bytes_per_sweep(w.N, sim.M, w.fp32)
    achieved = alg / (sweep_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": kernel, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg, "launch_ms": sweep_ms,
                "algorithmic_bytes_per_move": alg / moves_per_sweep,
                "share_of_step": S * sweep_ms / (ms / args.steps),
                "sweeps_on_tile_kernel": tile_sweeps, "sweeps_on_general_kernel": general_sweeps,
                "fused_floor_bytes_per_launch": fused_floor_bytes_per_sweep(w.N, sim.M, w.fp32),
                "state_bytes": state_bytes, "l2_bytes": l2_bytes,
                "note": ("one launch = one sweep; the state is L2-resident at this size (2 buffers x state_bytes < L2): the "
                         "load and shift phases run at the L2 bandwidth the SMs share, the sub-sweeps are bound by the FMA-class "
                         "pipes (see alu); the HBM fraction is reported because BASELINE.json names it")
                if 2 * state_bytes < l2_bytes else
                        ("one launch = one sweep; the state does not fit L2 (2 buffers x state_bytes > L2), so every sweep "
                         "streams it from and to HBM: `traffic` (ncu dram bytes per launch) against the fused floor "
                         "2 (e N + M) is the HBM figure")}
    if resident:
        roofline["launch_ms"] = sweep_ms * S
        roofline["sweep_ms"] = sweep_ms
        roofline["resident_ctas"] = cfg["resident_ctas"]
        roofline["algorithmic_bytes_per_launch"] = alg * S
        roofline["fused_floor_bytes_per_launch"] = 2.0 * state_bytes      # one launch reads the state once and writes it once
        roofline["note"] = (f"one launch of one cluster of {cfg['resident_ctas']} CTAs = all {S} sweeps of a step on the state "
                            "resident in shared memory: no HBM or L2 traffic inside the loop, the time is the latency of four "
                            "sub-sweeps + shift + six cluster barriers per sweep; `achieved` = the 7-pass algorithmic bytes of "
                            "those sweeps / launch time, reported because BASELINE.json names the HBM roofline")
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        try:
            tr = json.load(open(tpath))
            roofline["traffic"] = tr.get(f"{kernel}:{w.name}")
            ipl = tr.get(f"{kernel}:{w.name}:warp_instructions")
            if ipl and clocks.get("sm_mhz"):
                sms = torch.cuda.get_device_properties(dev).multi_processor_count
                issue_peak = sms * 4 * clocks["sm_mhz"] * 1e6          # warp instructions per second, 1 per scheduler per clock
                roofline["alu"] = {"bound": "alu", "achieved": ipl / (sweep_ms * 1e-3), "peak": issue_peak,
                                   "unit": "warp-instructions/s", "frac": ipl / (sweep_ms * 1e-3) / issue_peak,
                                   "warp_instructions_per_launch": ipl,
                                   "warp_instructions_per_move": ipl / moves_per_sweep}
        except Exception:
            pass

    # ---- max over ranks, whole-job aggregate ----
    ms, ms_e2e, moves, moves_e2e = aggregate(dist, dev, [ms, ms_e2e, moves, moves_e2e])
    value = moves / (ms * 1e-3)
    e2e = moves_e2e / (ms_e2e * 1e-3)

    cpu, cpu_strips = None, None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as O
        O.build()
        xy_cpu, _ = oracle_inputs(O, w)
        o = O.Oracle(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=w.fp32, w_target=w.w_target, disc=w.disc)
        o.load_positions(xy_cpu)
        o.sweep(1)
        a0 = o.acceptance()[0]
        t0 = time.perf_counter()
        o.sweep(args.cpu_baseline_sweeps)
        dt = time.perf_counter() - t0
        cpu = {"value": (o.acceptance()[0] - a0) / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{args.cpu_baseline_sweeps} sweeps of {w.name} (N={w.N}) after 1 warm-up sweep, "
                         f"single thread of {os.cpu_count()} host cores, {dt:.1f} s"}
        # the paper's multi-core CPU program: OpenMP, one horizontal strip of cells per thread, same
        # trajectory as the oracle bit for bit (checked here on the sample)
        O.build_strip()
        sb = O.StripBaseline(w.N, box, w.sigma, w.d, w.n_s, w.seed, fp32=w.fp32, w_target=w.w_target, disc=w.disc)
        sb.load_positions(xy_cpu)
        sb.sweep(1)
        b0 = sb.acceptance()[0]
        t0 = time.perf_counter()
        sb.sweep(args.cpu_baseline_sweeps)
        dts = time.perf_counter() - t0
        cpu_strips = {"value": (sb.acceptance()[0] - b0) / dts, "unit": UNIT, "cores": sb.threads, "kind": "openmp-strips",
                      "identical_to_oracle": sb.acceptance() == o.acceptance(),
                      "sample": f"the same {args.cpu_baseline_sweeps} sweeps, {sb.threads} OpenMP threads, {dts:.1f} s"}

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32" if w.fp32 else "f64", "data": "synthetic",
            "per_step": dict(spread(rates), unit=UNIT, note="this rank's steps; `value` is all steps' moves / all steps' time"),
            "config": dict(workload_config(w, S), parallelism=f"replicas x{world}" if world > 1 else "1 GPU",
                           l2="flushed between timed steps (256 MiB fill); the state itself is L2-resident",
                           step="load_positions + sweeps + contact histogram + get_positions + counters"),
            "clocks": clocks,
            "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": int(xy_pinned.numel() * 8),
                    "d2h_bytes_per_step": int(out_pinned.numel() * 8 + 20 * 8 + 64), "ms_per_step": ms_e2e / args.steps,
                    "per_step": spread(rates_e2e)},
            # cell-list build 4; one tile kernel per sweep (+ the general kernel's pass behind the 2-slot tile kernel: a
            # no-op unless a state was handed over), or one persistent launch without a tile kernel; histogram; unpack
            # (small systems: one launch of the cluster-resident kernel for all sweeps of a step)
            "gpu_launches": args.steps * (4 + (1 if cfg["resident_ctas"] else
                                               (S + (1 if cfg["tile_slots"] == 2 else 0) if cfg["tile_slots"] else 1)) + 1 + 1),
            "roofline": roofline,
            "cpu_baseline": cpu,
            "cpu_baseline_strips": cpu_strips,
            "paper_context": "PAPER.md L413: 1.09e9 trial moves/s on a Tesla K20 (different cell width, proposal and RNG)",
        }))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
