"""The five BASELINE.json configs as concrete synthetic workloads, plus small
random cases for property tests.  Parameters the configs omit are filled as SURVEY Q13 says
(marked "fill" below) and listed in DESIGN.md.
"""
from __future__ import annotations

import math
from typing import Optional

from . import collectives as C
from . import topologies as T
from .rng import SplitMix64, config_seed
from .types import (Collective, CollectiveBuilder, GpuCfg, Workload,
                    DEP_ACKED, DEP_DELIVERED, DEP_ISSUED)

LINE_BYTES = 128


def config1(cus: int = 4) -> Workload:
    """4 GPUs fully connected (1 line/cycle, 200 cycles); ring all-reduce of 1 MiB (8192 lines)
    in 4 chunks; C=4 (sweepable for pin P5), W=2, K=16, H=8; one design point."""
    w = Workload(name="config1")
    w.topologies.append(T.fully_connected(4, 256, 200))
    coll, _ = C.ring_allreduce(4, 8192, cus)
    w.collectives.append(coll)
    w.gpus.append(GpuCfg(cus, 2, 16, 8))
    w.points.append((0, 0, 0))
    w.meta.append({"algo": "ring", "lines": 8192})
    w.max_cycles = 1 << 22
    return w


def config2(sizes_log2_kib=range(6, 17)) -> Workload:
    """8 GPUs on one switch (4 lines/cycle per port, 150-cycle links, 50-cycle switch); ring and
    direct all-reduce over 64 KiB..64 MiB (11 sizes) -> 22 design points; C=64, W=4, K=32,
    H=16 (fill)."""
    w = Workload(name="config2")
    w.topologies.append(T.single_switch(8, 1024, 150, 50))
    w.gpus.append(GpuCfg(64, 4, 32, 16))
    for algo in ("ring", "direct"):
        for lk in sizes_log2_kib:
            m = (1 << lk) * 1024 // LINE_BYTES
            if algo == "ring":
                coll, _ = C.ring_allreduce(8, m, 64)
            else:
                coll = C.direct_allreduce(8, m, 64)
            w.collectives.append(coll)
            w.points.append((0, len(w.collectives) - 1, 0))
            w.meta.append({"algo": algo, "lines": m})
    w.max_cycles = 1 << 24
    return w


def config3(lines: int = 256 * 1024 * 1024 // LINE_BYTES) -> Workload:
    """64 GPUs = 8 nodes x 8; scale-up switch per node (4 lines/cycle), 2-level fat-tree
    scale-out (0.5 lines/cycle, 1000 cycles); hierarchical all-reduce of 256 MiB; C=128, W=8,
    K=32 (fill), H=16 (fill).  `lines` can be reduced for tests."""
    w = Workload(name="config3")
    w.topologies.append(T.nodes_fat_tree())
    w.collectives.append(C.hierarchical_allreduce(8, 8, lines, 128))
    w.gpus.append(GpuCfg(128, 8, 32, 16))
    w.points.append((0, 0, 0))
    w.meta.append({"algo": "hierarchical", "lines": lines})
    w.max_cycles = 1 << 26
    return w


_BW_CHOICES = (64, 128, 256, 512, 1024, 2048)
_ALGOS = ("ring", "direct", "dbt", "hd")


def config4_params(point: int) -> dict:
    """Draw the parameters of one design point of the config-4 sweep (no arrays are built).
    Draw order: topology bit, bandwidth, latency, algorithm, message bytes (log-uniform), CUs,
    wavefronts/CU, outstanding cap."""
    r = SplitMix64(config_seed(4, point))
    topo_kind = r.randint(0, 1)
    bw = _BW_CHOICES[r.randint(0, 5)]
    lat = r.randint(50, 2000)
    algo = _ALGOS[r.randint(0, 3)]
    u = r.uniform()
    nbytes = 4096.0 * math.exp(u * math.log(4096.0))       # 4 KiB .. 16 MiB
    m = max(16, int(math.ceil(nbytes / LINE_BYTES)))
    m = min(m, 16 * 1024 * 1024 // LINE_BYTES)
    cus = r.randint(8, 256)
    wpc = r.randint(1, 16)
    k = r.randint(4, 64)
    return {"topo": "ring16" if topo_kind == 0 else "torus4x4", "bw_q8": bw, "latency": lat,
            "algo": algo, "lines": m, "cus": cus, "wpc": wpc, "k": k}


def config4_point(point: int):
    """Build one design point of the config-4 sweep from its drawn parameters."""
    meta = config4_params(point)
    bw, lat, m, cus = meta["bw_q8"], meta["latency"], meta["lines"], meta["cus"]
    topo = T.ring(16, bw, lat) if meta["topo"] == "ring16" else T.torus2d(4, 4, bw, lat)
    algo = meta["algo"]
    if algo == "ring":
        coll, _ = C.ring_allreduce(16, m, cus)
    elif algo == "direct":
        coll = C.direct_allreduce(16, m, cus)
    elif algo == "dbt":
        coll = C.double_binary_tree_allreduce(16, m, cus)
    else:
        coll = C.halving_doubling_allreduce(16, m, cus)
    gpu = GpuCfg(cus, meta["wpc"], meta["k"], 32)       # H = 32 (fill)
    return topo, coll, gpu, meta


def config4(n_points: int = 4096, first: int = 0, indices=None) -> Workload:
    """Design-space sweep of 4096 seeded points on a 16-GPU ring / 4x4 torus (`indices`: only these
    points of the sweep, in the order given)."""
    w = Workload(name="config4")
    for p in (range(first, first + n_points) if indices is None else indices):
        topo, coll, gpu, meta = config4_point(p)
        w.topologies.append(topo)
        w.collectives.append(coll)
        w.gpus.append(gpu)
        i = len(w.topologies) - 1
        w.points.append((i, i, i))
        w.meta.append(meta)
    w.max_cycles = 1 << 26
    return w


def config5(n_nodes: int = 32, scale_lines: float = 1.0) -> Workload:
    """MoE-style all-to-all on 256 GPUs in a rail-optimized topology; per-pair sizes lognormal
    (median 32 KiB, sigma 1.0, clipped to [128 B, 4 MiB]); C=64, W=4, K=16, H=16 (fill).
    n_nodes / scale_lines shrink it for tests."""
    G = n_nodes * 8
    w = Workload(name="config5")
    w.topologies.append(T.rail_optimized(n_nodes=n_nodes))
    r = SplitMix64(config_seed(5, 0))
    table = {}
    for g in range(G):
        for d in range(G):
            if d == g:
                continue
            z = r.normal()
            nbytes = math.exp(math.log(32768.0) + 1.0 * z) * scale_lines
            table[(g, d)] = min(32768, max(1, int(math.ceil(nbytes / LINE_BYTES))))
    w.collectives.append(C.all_to_all(G, lambda g, d: table[(g, d)], 64))
    w.gpus.append(GpuCfg(64, 4, 16, 16))
    w.points.append((0, 0, 0))
    w.meta.append({"algo": "all_to_all", "lines": w.collectives[0].total_lines})
    w.max_cycles = 1 << 26
    return w


def by_name(name: str) -> Workload:
    return {"config1": config1, "config2": config2, "config3": config3,
            "config4": config4, "config5": config5}[name]()


# ----------------------------------------------------------------------------------------
# Small random cases for property tests (not part of BASELINE).
# ----------------------------------------------------------------------------------------

def random_topology(r: SplitMix64, n_gpus: int, n_switches: int):
    """Random strongly connected directed graph: a bidirectional spanning chain over all nodes
    in a shuffled order, plus random extra directed links; random bandwidth / latency."""
    V = n_gpus + n_switches
    order = list(range(V))
    for i in range(V - 1, 0, -1):
        j = r.randint(0, i)
        order[i], order[j] = order[j], order[i]
    bws = (64, 96, 128, 256, 384, 512, 1024)
    pairs = set()
    for i in range(V - 1):
        pairs.add((order[i], order[i + 1]))
        pairs.add((order[i + 1], order[i]))
    extra = r.randint(0, 2 * V)
    for _ in range(extra):
        a, b = r.randint(0, V - 1), r.randint(0, V - 1)
        if a != b:
            pairs.add((a, b))
    edges = [(a, b, bws[r.randint(0, len(bws) - 1)], r.randint(1, 40)) for (a, b) in sorted(pairs)]
    node_lat = [0] * n_gpus + [r.randint(0, 9) for _ in range(n_switches)]
    return T.Topology.from_edges(n_gpus, n_switches, node_lat, edges)


def random_collective(r: SplitMix64, n_gpus: int, cus: int, n_steps: int, max_lines: int) -> Collective:
    """Random step DAG with all three dependency kinds, honouring R3's locality rule."""
    b = CollectiveBuilder(n_gpus, "random")
    rows = []
    for s in range(n_steps):
        owner = r.randint(0, n_gpus - 1)
        dst = r.randint(0, n_gpus - 2)
        if dst >= owner:
            dst += 1
        lines = r.randint(1, max_lines)
        cu_lo = r.randint(0, cus - 1)
        cu_n = r.randint(1, cus - cu_lo)
        deps = []
        ndep = r.randint(0, 3)
        for _ in range(ndep):
            if s == 0:
                break
            p = r.randint(0, s - 1)
            kinds = []
            if rows[p][1] == owner:
                kinds.append(DEP_DELIVERED)
            if rows[p][0] == owner:
                kinds += [DEP_ACKED, DEP_ISSUED]
            if kinds and all(p != q for q, _ in deps):
                deps.append((p, kinds[r.randint(0, len(kinds) - 1)]))
        rows.append((owner, dst))
        b.add(owner, dst, lines, cu_lo, cu_n, deps)
    return b.build()


def random_workload(seed: int, n_points: int = 1, max_gpus: int = 4, max_switches: int = 2,
                    max_steps: int = 12, max_lines: int = 60) -> Workload:
    w = Workload(name=f"random{seed}")
    for p in range(n_points):
        r = SplitMix64(config_seed(9, seed * 1000 + p))
        g = r.randint(2, max_gpus)
        sw = r.randint(0, max_switches)
        topo = random_topology(r, g, sw)
        cus = r.randint(1, 6)
        gpu = GpuCfg(cus, r.randint(1, 4), r.randint(1, 9), r.randint(1, 6))
        coll = random_collective(r, g, cus, r.randint(1, max_steps), max_lines)
        w.topologies.append(topo); w.collectives.append(coll); w.gpus.append(gpu)
        w.points.append((p, p, p))
        w.meta.append({"seed": seed, "point": p})
    w.max_cycles = 1 << 22
    return w
