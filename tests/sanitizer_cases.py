"""Small runs of every per-sweep kernel family for `compute-sanitizer` (SURVEY.md section 5 "Race handling").

    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py

One tool per GPU call (B200_PROFILING.md).  Each case runs a few sweeps through the C ABI, with and without MPMC_DEBUG,
and compares the final state with the oracle so that a hazard that corrupts data also shows up as a mismatch.  The
summaries go to profiles/r2_sanitizer.md.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

from oracle import oracle as O  # noqa: E402
from paper_1211_1646_b200 import build, inputs as I  # noqa: E402
from paper_1211_1646_b200.binding import Mpmc  # noqa: E402


def run(name, N, box, xy, d, n_s, seed, fp32, sweeps, w_target=0.0, disc=False, want=None, resident=False):
    for debug in (True, False):
        o = O.Oracle(N, box, 1.0, d, n_s, seed, fp32=fp32, w_target=w_target, disc=disc)
        g = Mpmc(N, box, 1.0, d, n_s, seed, fp32=fp32, debug=debug, w_target=w_target, disc=disc, resident=resident)
        o.load_positions(xy)
        g.load_positions(torch.as_tensor(xy, device="cuda"))
        o.sweep(sweeps); g.sweep(sweeps)
        so, sg = o.debug_state(), g.debug_state()
        assert np.array_equal(so["counts"], sg["counts"]) and np.array_equal(so["ids"], sg["ids"])
        assert np.array_equal(so["slab"], sg["slab"]) and o.acceptance() == g.acceptance()
        hist = g.contact_histogram(0.005, 20)
        assert np.array_equal(hist, o.contact_histogram(0.005, 20))
        assert np.array_equal(g.get_positions().cpu().numpy(), o.get_positions())
        cfg, path = g.config(), g.path_sweeps()
        if want:
            for k, v in want.items():
                assert cfg[k] == v, (name, k, cfg)
        print(f"{name:28s} debug={int(debug)} fp{'32' if fp32 else '64'} N={N} cells={g.mx}x{g.my} tile_slots={cfg['tile_slots']} "
              f"tiles={cfg['ntx']}x{cfg['nty']} resident_ctas={cfg['resident_ctas'] if resident else 0} path={path} "
              f"max n={int(so['counts'].max())}  ok", flush=True)
        g.close()


def main():
    assert torch.cuda.is_available()
    build.build(); O.build()
    w = I.CONFIGS["C1"]
    xy, box = I.workload_inputs(w)
    for fp32 in (False, True):
        run("C1", w.N, box, xy, w.d, w.n_s, w.seed, fp32, 6, want={"tile_slots": 2})
        run("C1, cluster-resident", w.N, box, xy, w.d, w.n_s, w.seed, fp32, 6, resident=True)
    xy, box = I.jittered_lattice(50, 0.7, seed=50)                 # tiles of different sizes
    run("uneven tiling 50^2", 2500, box, xy, 0.15, 4, 50, True, 5, want={"tile_slots": 2})
    xy, box = I.jittered_lattice(50, 0.33, seed=50)                # ... with most cells empty
    run("uneven tiling, dilute", 2500, box, xy, 0.4, 4, 50, True, 5, want={"tile_slots": 2})
    xy, box = I.jittered_lattice(64, 0.50, seed=6)                 # cells with three disks on the 2-slot tile kernel
    run("three per cell, w=1.12", 4096, box, xy, 0.3, 4, 8, True, 40, w_target=1.12, want={"tile_slots": 2})
    run("three per cell, w=1.12", 4096, box, xy, 0.3, 8, 8, False, 20, w_target=1.12, want={"tile_slots": 2})
    xy, box = I.jittered_lattice(64, 0.6, seed=4)                  # general persistent kernel (n_s = 3)
    run("general kernel n_s=3", 4096, box, xy, 0.2, 3, 5, True, 5, want={"tile_slots": 0})
    w = I.CONFIGS["P256"]                                          # the paper's regime: 4-slot tile kernel, disc proposal
    xy, box = I.workload_inputs(w)
    run("P256", w.N, box, xy, w.d, w.n_s, w.seed, True, 3, w_target=w.w_target, disc=True, want={"tile_slots": 4})
    print("all cases identical to the oracle")


if __name__ == "__main__":
    main()
