"""Multi-process (gloo, world_size 2) test of the N>1 path's host logic: plan sharding and the
final gather. No GPU; each rank fills its shard with a deterministic function of the plan index."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2512_14098_b200 import shard
from paper_2512_14098_b200 import workloads as W


def test_plan_shard_partitions():
    for P in (1, 2, 7, 512, 4097):
        for world in (1, 2, 3, 8):
            ranges = [shard.plan_shard(P, r, world) for r in range(world)]
            assert ranges[0][0] == 0 and ranges[-1][1] == P
            assert all(a[1] == b[0] for a, b in zip(ranges, ranges[1:]))
            sizes = [e - b for b, e in ranges]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, P):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.config1_mllm(n_req=10, n_trials=1, n_rates=2, llm_max=4, e_steps=2)
        w.plans = w.plans.subset(np.arange(P))
        w.rate_mrps = w.rate_mrps[:P]
        s, idx = shard.shard_workload(w, rank, world)
        assert s.plans.n_plans == len(idx) and s.rate_mrps.shape[0] == len(idx)
        assert (s.plans.stage_c == w.plans.stage_c[idx]).all()
        local = torch.from_numpy(np.stack([idx * 10 + t for t in range(3)], axis=1).astype(np.int32))
        full = shard.gather_plan_results(local, P)
        want = np.stack([np.arange(P) * 10 + t for t in range(3)], axis=1)
        assert (full.numpy() == want).all()
        assert shard.best_plan(full) == P - 1
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("P", [5, 16])
def test_gather_world_size_2(P):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, P), nprocs=2, join=True)
