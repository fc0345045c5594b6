"""Plain containers for the flat integer arrays that cross the C-ABI (include/astra.h)."""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

# Dependency kinds: which timestamp of the producer step is waited on.
DEP_DELIVERED = 0   # producer's last line reached its dst   (requires dst(p) == owner(s))
DEP_ACKED = 1       # producer's last ack processed at owner (requires owner(p) == owner(s))
DEP_ISSUED = 2      # producer's last line issued            (requires owner(p) == owner(s))


def _u32(x) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(x, dtype=np.int64))
    if a.size and (a.min() < 0 or a.max() > 0xFFFFFFFF):
        raise ValueError("value out of uint32 range")
    return a.astype(np.uint32)


@dataclass
class Topology:
    """InfraGraph flattened to CSR by TAIL node.

    Nodes 0..n_gpus-1 are GPUs (node id == rank), then the switches.  Link id ==
    CSR position; heads strictly ascending inside a row.  bw_q8 = lines/cycle*256.
    """
    n_gpus: int
    n_switches: int
    node_latency: np.ndarray   # [V] u32
    row_ptr: np.ndarray        # [V+1] u32
    head: np.ndarray           # [E] u32
    bw_q8: np.ndarray          # [E] u32
    latency: np.ndarray        # [E] u32

    @property
    def n_nodes(self) -> int:
        return self.n_gpus + self.n_switches

    @property
    def n_links(self) -> int:
        return int(self.head.shape[0])

    @staticmethod
    def from_edges(n_gpus: int, n_switches: int, node_latency, edges) -> "Topology":
        """edges: iterable of (tail, head, bw_q8, latency); sorted here into CSR order."""
        V = n_gpus + n_switches
        es = sorted((int(t), int(h), int(b), int(l)) for (t, h, b, l) in edges)
        row_ptr = np.zeros(V + 1, dtype=np.int64)
        for t, _, _, _ in es:
            row_ptr[t + 1] += 1
        row_ptr = np.cumsum(row_ptr)
        return Topology(
            n_gpus=n_gpus, n_switches=n_switches,
            node_latency=_u32(node_latency),
            row_ptr=_u32(row_ptr),
            head=_u32([e[1] for e in es]),
            bw_q8=_u32([e[2] for e in es]),
            latency=_u32([e[3] for e in es]),
        )

    def tail(self) -> np.ndarray:
        t = np.zeros(self.n_links, dtype=np.uint32)
        for v in range(self.n_nodes):
            t[self.row_ptr[v]:self.row_ptr[v + 1]] = v
        return t

    def link_id(self, tail: int, head: int) -> int:
        lo, hi = int(self.row_ptr[tail]), int(self.row_ptr[tail + 1])
        for e in range(lo, hi):
            if int(self.head[e]) == head:
                return e
        raise KeyError((tail, head))


@dataclass
class Collective:
    """Per-GPU step DAG: step s = owner sends `lines` 128 B lines to dst
    using CUs [cu_lo, cu_lo+cu_n) of the owner; deps as CSR with kinds."""
    n_gpus: int
    owner: np.ndarray
    dst: np.ndarray
    lines: np.ndarray
    cu_lo: np.ndarray
    cu_n: np.ndarray
    dep_ptr: np.ndarray
    dep_step: np.ndarray
    dep_kind: np.ndarray   # u8
    name: str = ""

    @property
    def n_steps(self) -> int:
        return int(self.owner.shape[0])

    @property
    def total_lines(self) -> int:
        return int(self.lines.astype(np.uint64).sum())


class CollectiveBuilder:
    def __init__(self, n_gpus: int, name: str = ""):
        self.n_gpus = n_gpus
        self.name = name
        self.rows: List[Tuple[int, int, int, int, int, List[Tuple[int, int]]]] = []

    def add(self, owner, dst, lines, cu_lo, cu_n, deps=()) -> int:
        sid = len(self.rows)
        deps = [(int(p), int(k)) for (p, k) in deps]
        for p, _ in deps:
            if not (0 <= p < sid):
                raise ValueError("dep id must be < step id")
        self.rows.append((int(owner), int(dst), int(lines), int(cu_lo), int(cu_n), deps))
        return sid

    def build(self) -> Collective:
        dep_ptr = [0]
        dep_step: List[int] = []
        dep_kind: List[int] = []
        for r in self.rows:
            for p, k in r[5]:
                dep_step.append(p)
                dep_kind.append(k)
            dep_ptr.append(len(dep_step))
        return Collective(
            n_gpus=self.n_gpus,
            owner=_u32([r[0] for r in self.rows]),
            dst=_u32([r[1] for r in self.rows]),
            lines=_u32([r[2] for r in self.rows]),
            cu_lo=_u32([r[3] for r in self.rows]),
            cu_n=_u32([r[4] for r in self.rows]),
            dep_ptr=_u32(dep_ptr),
            dep_step=_u32(dep_step),
            dep_kind=np.ascontiguousarray(np.asarray(dep_kind, dtype=np.uint8)),
            name=self.name,
        )


GPU_ISSUE_PER_CU = 1    # a CU dispatches at most one line per cycle (lowest ready wavefront)
GPU_CAP_PER_CU = 2      # max_outstanding bounds the CU's wavefronts together


@dataclass
class GpuCfg:
    """astra_set_gpu parameters (PAPER.md:L189 CUs, L165 wavefronts, L209/L297 outstanding cap,
    L221 memory channels -> HBM rate)."""
    cus: int
    wavefronts_per_cu: int
    max_outstanding: int          # per wavefront -- per CU when mode & GPU_CAP_PER_CU
    hbm_lines_per_cycle: int
    mode: int = 0                 # GPU_ISSUE_PER_CU | GPU_CAP_PER_CU: the paper's per-CU readings


@dataclass
class Workload:
    """A batch: tables of topologies / collectives / GPU configs and the design points
    (topo index, collective index, gpu index) that reference them."""
    name: str
    topologies: List[Topology] = field(default_factory=list)
    collectives: List[Collective] = field(default_factory=list)
    gpus: List[GpuCfg] = field(default_factory=list)
    points: List[Tuple[int, int, int]] = field(default_factory=list)
    max_cycles: int = 1 << 31
    meta: List[dict] = field(default_factory=list)   # per point, free-form description

    @property
    def n_points(self) -> int:
        return len(self.points)

    def total_lines(self) -> int:
        return sum(self.collectives[c].total_lines for (_, c, _) in self.points)

    def point(self, i: int) -> Tuple[Topology, Collective, GpuCfg]:
        t, c, g = self.points[i]
        return self.topologies[t], self.collectives[c], self.gpus[g]

    def subset(self, idx) -> "Workload":
        """A workload holding only the listed points (tables re-indexed, order kept)."""
        w = Workload(name=f"{self.name}[subset]", max_cycles=self.max_cycles)
        tmap, cmap, gmap = {}, {}, {}
        for i in idx:
            t, c, g = self.points[i]
            if t not in tmap:
                tmap[t] = len(w.topologies); w.topologies.append(self.topologies[t])
            if c not in cmap:
                cmap[c] = len(w.collectives); w.collectives.append(self.collectives[c])
            if g not in gmap:
                gmap[g] = len(w.gpus); w.gpus.append(self.gpus[g])
            w.points.append((tmap[t], cmap[c], gmap[g]))
            w.meta.append(self.meta[i] if i < len(self.meta) else {})
        return w
