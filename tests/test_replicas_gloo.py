"""Multi-GPU is "replicas only": N independent simulations, no data-path
collective.  The only distributed logic is the report: MAX over ranks of the device times, SUM over ranks of the
moves (bench.aggregate).  Covered here with world_size 2 on gloo, CPU only."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r: 10 + r ms resident, 20 - r ms end to end, (r + 1) * 1000 moves, (r + 1) * 500 moves end to end
    got = bench.aggregate(dist, torch.device("cpu"), [10.0 + rank, 20.0 - rank, (rank + 1) * 1000.0, (rank + 1) * 500.0])
    dist.barrier()
    if rank == 0:
        torch.save(got, out)
    dist.destroy_process_group()


def test_aggregate_takes_max_time_and_sum_of_moves(tmp_path):
    out = str(tmp_path / "agg.pt")
    port = 29500 + (os.getpid() % 2000)
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    ms, ms_e2e, moves, moves_e2e = torch.load(out)
    assert ms == 11.0 and ms_e2e == 20.0            # slowest rank
    assert moves == 3000.0 and moves_e2e == 1500.0  # all ranks


def test_aggregate_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(None, None, [1.0, 2.0, 3.0, 4.0]) == [1.0, 2.0, 3.0, 4.0]


def test_replica_seeds_differ():
    """bench.py gives replica r the seed config.seed + r: their streams must differ (here: the oracle's draws)."""
    sys.path.insert(0, ROOT)
    from oracle import oracle as O
    O.build()
    a = O.sweep_draws(1, 0), O.sweep_draws(1, 1), O.sweep_draws(1, 2)
    b = O.sweep_draws(2, 0), O.sweep_draws(2, 1), O.sweep_draws(2, 2)
    assert a != b
