"""Host logic of bench.py's N > 1 path ("replicas only"), on CPU with gloo, world_size 2:
the job's device time is the max over ranks and the value aggregates every rank's replica."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import rte_workloads as wl
    cfg = wl.CONFIGS["cfg2"]
    my_ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    dist.barrier()
    ms = bench.max_over_ranks(my_ms, dist, torch.device("cpu"))
    value = bench.job_value(cfg, 7, world, ms)
    out[rank] = (ms, value)
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_world_size_2():
    import bench
    import rte_workloads as wl
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    cfg = wl.CONFIGS["cfg2"]
    for rank in range(world):
        ms, value = res[rank]
        assert ms == 15.0                                        # the slowest rank's time, on every rank
        assert abs(value - cfg.C * cfg.G * 7 * 2 / 15e-3) <= 1e-6 * value
    # single process: no collective, value of one replica
    assert bench.max_over_ranks(3.5, None, None) == 3.5
    assert abs(bench.job_value(cfg, 7, 1, 3.5) - cfg.C * cfg.G * 7 / 3.5e-3) < 1.0


def test_algorithmic_bytes_model():
    """8 S + 12 G bytes per 3-D step, 5 S + 12 G per 2-D step; x pass 2 S + maps, others 3 S."""
    import bench
    import rte_workloads as wl
    for name, cfg in wl.CONFIGS.items():
        S = 4 * cfg.C * cfg.G
        per_axis, per_step = bench.algorithmic_bytes(cfg)
        assert per_axis[0] == 2 * S + 12 * cfg.G and per_axis[1] == 3 * S
        assert per_step == (8 if cfg.dim == 3 else 5) * S + 12 * cfg.G
