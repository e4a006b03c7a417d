"""Multi-GPU arrangement of the hot path = replicas only.  World-size-2 gloo test of the
host logic bench.py uses under torchrun: per-rank seeds give independent input streams, `value` is the total
work over the slowest rank's time, and no data-path collective exists (only scalar timing reductions)."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2606_15476_b200 import scenes as S
    sc = S.StressScene(n_batches=1, frames_per_batch=1, n_objects=60, seed=S.get_config(4).seed + bench.rank_seed(0, rank))
    fr = sc.batch(0)[0]
    digest = float(np.asarray(fr.depth, np.float64).sum())
    frames_local, ms_local = 16 * (rank + 1), 10.0 * (rank + 1)        # rank 1 is slower and did more
    value, total, ms = bench.aggregate_throughput(frames_local, ms_local, world)
    digests = [None] * world
    dist.all_gather_object(digests, digest)
    out[rank] = (value, total, ms, digests)
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_world_size_2_gloo():
    world = 2
    port = _free_port()
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        value, total, ms, digests = res[rank]
        assert total == 48 and ms == 20.0 and abs(value - 48 / 20e-3) < 1e-9      # total frames / max time
        assert digests[0] != digests[1]                                          # independent input streams
    assert res[0][3] == res[1][3]
