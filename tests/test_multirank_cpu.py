"""-m "not gpu": the N > 1 host logic of bench.py on CPU with gloo, world_size 2: every rank gets its
own shard (same recipe, different seed, no data-path collective) and the only exchange is
MAX(time) / SUM(units).  Multi-GPU decomposition: DESIGN.md "Multi-GPU"."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_1605_07023_b200 import synth
    cfg = bench.rank_config(synth.shrink(synth.get_config("cfg1"), n_ant=6, n_times=8, n_chan=4, grid_size=256), rank)
    wl = synth.make_workload(cfg)
    times, total = bench.reduce_over_ranks([10.0 + rank, 5.0 - rank], 1000 * (rank + 1), torch.device("cpu"), world)
    out.put((rank, cfg.seed, float(np.abs(wl.vis).sum()), times, total))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, v0, t0, tot0), (r1, s1, v1, t1, tot1) = res
    assert s0 != s1 and v0 != v1                       # different shards
    assert t0 == t1 == [11.0, 5.0]                     # max over ranks
    assert tot0 == tot1 == 3000.0                      # whole-job units
