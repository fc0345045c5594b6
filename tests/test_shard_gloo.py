"""The N > 1 path: a batch shards by design point, no collective on the data path.
World-size-2 gloo run on CPU: each rank simulates its share (the per-point simulator is injected;
here the CPU oracle stands in for the engine, which needs a GPU) and the shares are gathered."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

from astra_inputs import configs
from paper_2606_10440_b200.shard import point_costs, run_sharded, shard_points


def test_shard_points_is_a_partition_and_balanced():
    costs = [5.0, 1.0, 9.0, 3.0, 3.0, 7.0, 2.0]
    for world in (1, 2, 3, 8):
        shards = shard_points(costs, world)
        assert sorted(i for s in shards for i in s) == list(range(len(costs)))
        loads = [sum(costs[i] for i in s) for s in shards]
        assert max(loads) <= sum(costs) / world + max(costs)          # LPT bound
    assert shard_points(costs, 2) == shard_points(costs, 2)           # deterministic
    assert shard_points([], 3) == [[], [], []]


def _oracle_sim(workload, indices):
    from oracle import oracle
    res = oracle.run_workload(workload, list(indices), processes=1, flags=oracle.FLAG_PRUNED_SCAN)
    return [(r.status, int(r.completion), r.step_ts.copy(), r.link_lines.copy()) for r in res]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = configs.random_workload(17, n_points=7, max_gpus=5, max_steps=16, max_lines=120)
    merged = run_sharded(w, _oracle_sim, rank, world)
    np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([m[1] for m in merged], dtype=np.int64))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_gloo(tmp_path):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    w = configs.random_workload(17, n_points=7, max_gpus=5, max_steps=16, max_lines=120)
    single = run_sharded(w, _oracle_sim, 0, 1)
    want = np.array([m[1] for m in single], dtype=np.int64)
    for r in range(2):
        got = np.load(os.path.join(str(tmp_path), f"r{r}.npy"))
        assert (got == want).all()                                   # every rank holds every point's result
    assert len(point_costs(w)) == w.n_points
