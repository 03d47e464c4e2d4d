"""N > 1 path of bench.py on CPU: the queue is sharded by rank (disjoint, covering id ranges), no collective on the
data path; the per-rank counts are summed and the per-rank times maxed exactly as bench.py does, over gloo with
world_size 2."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_26341_b200 import workloads as wl
import bench


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, P, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    first = bench.shard_first_id(rank, P)
    d, theta, x0 = wl.generate(0, P, first_id=first)
    # stand-ins for the per-rank results of a solve: what rank r would report
    solved, iters, ms = float(P - rank), float(10 * P + rank), 5.0 + rank
    red = torch.tensor([ms], dtype=torch.float64)
    cnt = torch.tensor([solved, iters, float(P)], dtype=torch.float64)
    bench.reduce_over_ranks(red, cnt, world)
    ids = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(ids, torch.tensor([first], dtype=torch.int64))
    chk = torch.tensor([float(theta.sum())], dtype=torch.float64)
    sums = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(sums, chk)
    if rank == 0:
        np.save(out, np.array([red[0].item(), *cnt.tolist(), *[i.item() for i in ids], *[v.item() for v in sums]]))
    dist.destroy_process_group()


def test_queue_sharding_and_reduction_world_size_2(tmp_path):
    P, world = 8, 2
    out = str(tmp_path / "r.npy")
    mp.spawn(_worker, args=(world, _free_port(), P, out), nprocs=world, join=True)
    r = np.load(out)
    assert r[0] == 6.0                       # max over ranks of the step time
    assert r[1] == (P - 0) + (P - 1)         # solved counts summed
    assert r[2] == 10 * P + 10 * P + 1       # iterations summed
    assert r[3] == world * P                 # problems summed: whole-job aggregate
    assert list(r[4:6]) == [0, P]            # disjoint, contiguous id ranges
    # the shards are exactly the rows a single process would generate
    d, theta, _ = wl.generate(0, world * P)
    assert np.isclose(r[6], theta[:P].sum()) and np.isclose(r[7], theta[P:].sum())
