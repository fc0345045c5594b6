"""NoC-level GPU model (section 5.1 "Target GPU Architecture"):
every GPU is an 8 x 4 mesh of 32 routers with four CUs each (128 CUs), 16 memory channels on each of the
16 routers of the top and bottom rows (256 channels) and four I/O ports on each of the 8 routers of the
left and right columns (32 ports): 448 nodes per GPU.  CUs and memory channels are the simulator's
endpoints ("GPUs" of the C-ABI: the nodes that own steps and receive lines), routers and I/O ports are
switches; the scale-up fabric joins I/O port p of every GPU through switch p.

Inputs only: the graph and a CU-level collective on it; no routing, no timing.

Readings (the paper gives bandwidths and one latency, no clock and no on-chip latencies; 1 cycle is
taken as about 1 ns and every value as the nearest power of two, "power-of-two
configuration values"): on-chip links 1 TiB/s -> 8 lines/cycle; 4 TiB/s over 256 memory channels -> 1/8
line/cycle per channel; 1 TiB/s over 32 I/O ports -> 1/4 line/cycle per port, scale-up link latency
1 us -> 1024 cycles; mesh hop, CU attach and I/O attach latency 4 cycles, memory channel 64 cycles
(our fills).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List

from .types import Collective, CollectiveBuilder, Topology, DEP_DELIVERED

ROWS, COLS = 4, 8
CUS_PER_ROUTER, CH_PER_EDGE_ROUTER, IO_PER_SIDE_ROUTER = 4, 16, 4
N_CU, N_CH, N_IO, N_ROUTER = 128, 256, 32, 32
ENDPOINTS_PER_GPU = N_CU + N_CH              # CUs and memory channels: the simulator's "GPU" nodes
NODES_PER_GPU = ENDPOINTS_PER_GPU + N_ROUTER + N_IO     # 448


@dataclass
class NocMap:
    """Node ids of a NoC cluster: endpoints first (per GPU: CUs, then memory channels), then per GPU its
    routers and I/O ports, then the scale-up switches."""
    n_gpus: int

    def cu(self, g: int, c: int) -> int:
        return g * ENDPOINTS_PER_GPU + c

    def channel(self, g: int, ch: int) -> int:
        return g * ENDPOINTS_PER_GPU + N_CU + ch

    def router(self, g: int, r: int, c: int) -> int:
        return self.n_gpus * ENDPOINTS_PER_GPU + g * (N_ROUTER + N_IO) + r * COLS + c

    def io(self, g: int, p: int) -> int:
        return self.n_gpus * ENDPOINTS_PER_GPU + g * (N_ROUTER + N_IO) + N_ROUTER + p

    def fabric(self, p: int) -> int:
        return self.n_gpus * NODES_PER_GPU + p

    def cu_router(self, c: int):
        r = c // CUS_PER_ROUTER
        return r // COLS, r % COLS

    def channel_router(self, ch: int):
        r = ch // CH_PER_EDGE_ROUTER                  # 0..7 top row, 8..15 bottom row
        return (0, r) if r < COLS else (ROWS - 1, r - COLS)

    def io_router(self, p: int):
        r = p // IO_PER_SIDE_ROUTER                   # 0..3 left column, 4..7 right column
        return (r, 0) if r < ROWS else (r - ROWS, COLS - 1)


def noc_cluster(n_gpus: int, mesh_bw_q8: int = 2048, mesh_lat: int = 4, cu_lat: int = 4,
                ch_bw_q8: int = 32, ch_lat: int = 64, io_bw_q8: int = 64, io_lat: int = 4,
                link_lat: int = 1024):
    """The graph of `n_gpus` NoC-level GPUs and their scale-up fabric.  Returns (Topology, NocMap)."""
    m = NocMap(n_gpus)
    edges = []

    def both(a, b, bw, lat):
        edges.append((a, b, bw, lat)); edges.append((b, a, bw, lat))

    for g in range(n_gpus):
        for r in range(ROWS):
            for c in range(COLS):
                if c + 1 < COLS:
                    both(m.router(g, r, c), m.router(g, r, c + 1), mesh_bw_q8, mesh_lat)
                if r + 1 < ROWS:
                    both(m.router(g, r, c), m.router(g, r + 1, c), mesh_bw_q8, mesh_lat)
        for cu in range(N_CU):
            both(m.cu(g, cu), m.router(g, *m.cu_router(cu)), mesh_bw_q8, cu_lat)
        for ch in range(N_CH):
            both(m.channel(g, ch), m.router(g, *m.channel_router(ch)), ch_bw_q8, ch_lat)
        for p in range(N_IO):
            both(m.io(g, p), m.router(g, *m.io_router(p)), io_bw_q8, io_lat)
            both(m.io(g, p), m.fabric(p), io_bw_q8, link_lat)
    n_end = n_gpus * ENDPOINTS_PER_GPU
    n_sw = n_gpus * (N_ROUTER + N_IO) + N_IO
    return Topology.from_edges(n_end, n_sw, [0] * (n_end + n_sw), edges), m


def noc_all_gather(m: NocMap, lines_per_gpu: int, workgroups: int = 32, channels_per_wg: int = 4,
                   local_load: bool = True) -> Collective:
    """CU-level direct all-gather ("All-Gather ... with 32 work-groups per GPU"): workgroup w of
    GPU g (on CU w * 128 / workgroups) copies slice w of g's buffer to every other GPU, a MemcpyOp per (peer,
    memory channel): the slice is interleaved over `channels_per_wg` channels (channel (w * channels_per_wg
    + j) mod 256 on both sides).  With local_load the data first comes out of g's own memory: a one-line
    request from the CU to the local channel, the channel's response to the CU (PAPER.md:L150 MemcpyOp = Load,
    Waitcnt, Store; one request per (peer, channel) chunk: the get reading of collectives.as_get), and the
    remote store waits for that response."""
    n = m.n_gpus
    b = CollectiveBuilder(n * ENDPOINTS_PER_GPU, f"noc_all_gather_n{n}_m{lines_per_gpu}")
    per_wg = [lines_per_gpu // workgroups + (1 if w < lines_per_gpu % workgroups else 0) for w in range(workgroups)]
    for g in range(n):
        for w in range(workgroups):
            cu = m.cu(g, w * N_CU // workgroups)
            for p in range(1, n):
                peer = (g + p) % n
                for j in range(channels_per_wg):
                    lines = per_wg[w] // channels_per_wg + (1 if j < per_wg[w] % channels_per_wg else 0)
                    if lines == 0:
                        continue
                    ch = (w * channels_per_wg + j) % N_CH
                    deps = []
                    if local_load:
                        req = b.add(cu, m.channel(g, ch), 1, 0, 1)
                        resp = b.add(m.channel(g, ch), cu, lines, 0, 1, [(req, DEP_DELIVERED)])
                        deps = [(resp, DEP_DELIVERED)]
                    b.add(cu, m.channel(peer, ch), lines, 0, 1, deps)
    return b.build()
