"""N > 1 host logic (bench.py): events shard across ranks with no data-path collective; the job time is the max
over ranks.  Two gloo processes on CPU; the oracle stands in for the device path."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import bench
    import oracle
    import pixgen
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    seeds = bench.shard_seeds(2, rank)
    det = pixgen.detector("tiny")
    batch = pixgen.events(det, "tiny", seeds)
    n_clusters = 0
    for e in range(batch.n_events):
        o = oracle.process(det, *batch.event(e), bench.PARAMS, max_clusters_per_event=1 << 16)
        n_clusters += int(o["summary"][14])
    ms = bench.max_over_ranks(10.0 * (rank + 1), dist)          # slowest rank decides
    tot = torch.tensor([n_clusters, len(batch.words)], dtype=torch.int64)
    dist.all_reduce(tot)                                          # optional 16-counter style summary sum
    out[rank] = (seeds.tolist(), ms, tot.tolist(), n_clusters)
    dist.destroy_process_group()


def test_two_ranks_shard_events_and_reduce_max():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    s0, s1 = set(res[0][0]), set(res[1][0])
    assert s0.isdisjoint(s1) and len(s0) == len(s1) == 2          # disjoint shards, equal work per rank (weak scaling)
    assert res[0][1] == res[1][1] == 20.0                         # max over ranks
    assert res[0][2] == res[1][2]
    assert res[0][2][0] == res[0][3] + res[1][3] and res[0][3] > 0 and res[1][3] > 0
