"""Topology builders (InfraGraph-style graphs flattened to CSR).

Every builder returns a `Topology`.  Bandwidth is in lines/cycle * 256 (bw_q8), latency in
cycles.  Switch traversal cost is a per-node latency.
"""
from __future__ import annotations

from .types import Topology


def fully_connected(n_gpus: int, bw_q8: int, latency: int) -> Topology:
    """BASELINE config 1: every ordered GPU pair has a direct link."""
    edges = [(a, b, bw_q8, latency) for a in range(n_gpus) for b in range(n_gpus) if a != b]
    return Topology.from_edges(n_gpus, 0, [0] * n_gpus, edges)


def single_switch(n_gpus: int, bw_q8: int, link_latency: int, switch_latency: int) -> Topology:
    """BASELINE config 2: one scale-up switch, one port per GPU (the paper's SingleTierFabric
    shape)."""
    sw = n_gpus
    edges = []
    for g in range(n_gpus):
        edges.append((g, sw, bw_q8, link_latency))
        edges.append((sw, g, bw_q8, link_latency))
    return Topology.from_edges(n_gpus, 1, [0] * n_gpus + [switch_latency], edges)


def ring(n_gpus: int, bw_q8: int, latency: int) -> Topology:
    """Bidirectional ring g <-> g+-1 (config 4)."""
    edges = set()
    for g in range(n_gpus):
        for h in ((g + 1) % n_gpus, (g - 1) % n_gpus):
            if h != g:
                edges.add((g, h))
    return Topology.from_edges(n_gpus, 0, [0] * n_gpus,
                               [(a, b, bw_q8, latency) for (a, b) in sorted(edges)])


def torus2d(rows: int, cols: int, bw_q8: int, latency: int) -> Topology:
    """rows x cols 2D torus with wrap-around in both dimensions (config 4)."""
    n = rows * cols
    edges = set()
    for r in range(rows):
        for c in range(cols):
            g = r * cols + c
            for (rr, cc) in ((r, (c + 1) % cols), (r, (c - 1) % cols),
                             ((r + 1) % rows, c), ((r - 1) % rows, c)):
                h = rr * cols + cc
                if h != g:
                    edges.add((g, h))
    return Topology.from_edges(n, 0, [0] * n,
                               [(a, b, bw_q8, latency) for (a, b) in sorted(edges)])


def nodes_fat_tree(n_nodes: int = 8, gpus_per_node: int = 8, n_spines: int = 4,
                   scaleup_bw_q8: int = 1024, scaleup_latency: int = 150,
                   scaleup_switch_latency: int = 50,
                   scaleout_bw_q8: int = 128, scaleout_latency: int = 1000,
                   scaleout_switch_latency: int = 0) -> Topology:
    """BASELINE config 3: per-node scale-up switch plus a 2-level fat-tree scale-out
    (one leaf per node, every leaf wired to every spine; the ClosFatTreeFabric shape of
    PAPER.md:L247).  Node ids: GPUs, node switches, leaves, spines."""
    G = n_nodes * gpus_per_node
    nsw0 = G
    leaf0 = G + n_nodes
    spine0 = leaf0 + n_nodes
    n_sw = n_nodes + n_nodes + n_spines
    node_lat = [0] * G + [scaleup_switch_latency] * n_nodes + \
        [scaleout_switch_latency] * (n_nodes + n_spines)
    edges = []
    for g in range(G):
        nd = g // gpus_per_node
        edges.append((g, nsw0 + nd, scaleup_bw_q8, scaleup_latency))
        edges.append((nsw0 + nd, g, scaleup_bw_q8, scaleup_latency))
        edges.append((g, leaf0 + nd, scaleout_bw_q8, scaleout_latency))
        edges.append((leaf0 + nd, g, scaleout_bw_q8, scaleout_latency))
    for nd in range(n_nodes):
        for s in range(n_spines):
            edges.append((leaf0 + nd, spine0 + s, scaleout_bw_q8, scaleout_latency))
            edges.append((spine0 + s, leaf0 + nd, scaleout_bw_q8, scaleout_latency))
    return Topology.from_edges(G, n_sw, node_lat, edges)


def rail_optimized(n_nodes: int = 32, gpus_per_node: int = 8,
                   scaleup_bw_q8: int = 1024, scaleup_latency: int = 150,
                   scaleup_switch_latency: int = 50,
                   rail_bw_q8: int = 256, rail_latency: int = 800,
                   rail_switch_latency: int = 0) -> Topology:
    """BASELINE config 5: per-node scale-up switch plus one rail switch per local index
    (rail r joins local GPU r of every node).  Node ids: GPUs, node switches, rail switches."""
    G = n_nodes * gpus_per_node
    nsw0 = G
    rail0 = G + n_nodes
    node_lat = [0] * G + [scaleup_switch_latency] * n_nodes + [rail_switch_latency] * gpus_per_node
    edges = []
    for g in range(G):
        nd, loc = divmod(g, gpus_per_node)
        edges.append((g, nsw0 + nd, scaleup_bw_q8, scaleup_latency))
        edges.append((nsw0 + nd, g, scaleup_bw_q8, scaleup_latency))
        edges.append((g, rail0 + loc, rail_bw_q8, rail_latency))
        edges.append((rail0 + loc, g, rail_bw_q8, rail_latency))
    return Topology.from_edges(G, n_nodes + gpus_per_node, node_lat, edges)


def line(n_gpus: int, bw_q8: int, latency: int) -> Topology:
    """Bidirectional chain 0-1-...-(n-1); used by tests (multi-hop GPU transit)."""
    edges = []
    for g in range(n_gpus - 1):
        edges.append((g, g + 1, bw_q8, latency))
        edges.append((g + 1, g, bw_q8, latency))
    return Topology.from_edges(n_gpus, 0, [0] * n_gpus, edges)
