"""Multi-GPU use of the engine: design points are independent (R1), so a batch shards by design
point with no collective on the data path.  One process per GPU; every rank runs
its own astra_ctx on its share and the few KB of results per point are gathered on the host side
with torch.distributed (gloo or nccl object gather) -- plumbing, not part of the simulation.

A single design point does not shard across GPUs ("replicas only").
"""
from __future__ import annotations

from typing import List, Sequence


def point_costs(workload) -> List[float]:
    """Cost proxy of every design point: lines issued x (1 + GPUs/16).  Only the order matters."""
    out = []
    for (t, c, _g) in workload.points:
        coll = workload.collectives[c]
        out.append(float(coll.total_lines) * (1.0 + workload.topologies[t].n_gpus / 16.0))
    return out


def shard_points(costs: Sequence[float], world_size: int) -> List[List[int]]:
    """Longest-processing-time-first greedy: points by decreasing cost, each to the least loaded
    rank (ties: lowest rank).  Deterministic; every rank computes the same partition."""
    if world_size < 1:
        raise ValueError("world_size must be >= 1")
    order = sorted(range(len(costs)), key=lambda i: (-costs[i], i))
    load = [0.0] * world_size
    shards: List[List[int]] = [[] for _ in range(world_size)]
    for i in order:
        r = min(range(world_size), key=lambda j: (load[j], j))
        shards[r].append(i)
        load[r] += costs[i]
    for s in shards:
        s.sort()
    return shards


def run_sharded(workload, simulate, rank: int, world_size: int, gather=None, costs=None):
    """Run this rank's share of `workload` through `simulate(workload, indices) -> list of per-point
    results` and gather all shares.  `gather(obj) -> list of one obj per rank` defaults to
    torch.distributed.all_gather_object on the default process group (world_size > 1).
    `costs` (one per point) replaces point_costs(workload); `workload` then only needs `n_points`,
    so a rank can build just its own points inside `simulate`.
    Returns the results of ALL points in workload order (on every rank)."""
    shards = shard_points(point_costs(workload) if costs is None else costs, world_size)
    mine = shards[rank]
    local = simulate(workload, mine) if mine else []
    if len(local) != len(mine):
        raise RuntimeError("simulate() returned a wrong number of results")
    if world_size == 1:
        parts = [list(zip(mine, local))]
    else:
        if gather is None:
            import torch.distributed as dist

            def gather(obj):
                out = [None] * world_size
                dist.all_gather_object(out, obj)
                return out
        parts = gather(list(zip(mine, local)))
    merged = [None] * workload.n_points
    for part in parts:
        for i, res in part:
            if merged[i] is not None:
                raise RuntimeError(f"design point {i} simulated twice")
            merged[i] = res
    if any(m is None for m in merged):
        raise RuntimeError("a design point was not simulated by any rank")
    return merged
