"""NoC-level GPU model: the generator astra_inputs/noc.py at reduced scale,
run through the unchanged oracle and engine (CUs and memory channels are the endpoints, routers and I/O ports the
switches)."""
import numpy as np
import pytest

from astra_inputs import GpuCfg, Workload, noc
from astra_inputs.types import CollectiveBuilder
from oracle import oracle


def _single(topo, coll, gpu, max_cycles=1 << 24):
    w = Workload(name=coll.name or "noc", max_cycles=max_cycles)
    w.topologies.append(topo); w.collectives.append(coll); w.gpus.append(gpu)
    w.points.append((0, 0, 0)); w.meta.append({})
    return w


def test_noc_structure():
    """32 routers, 128 CUs, 256 memory channels, 32 I/O ports = 448 nodes per GPU; 4 TiB/s of memory and
    1 TiB/s of scale-up bandwidth against 1 TiB/s on-chip links."""
    for n in (1, 2, 4):
        t, m = noc.noc_cluster(n)
        assert noc.NODES_PER_GPU == 448
        assert t.n_gpus == n * 384 and t.n_switches == n * 64 + 32 and t.n_nodes == n * 448 + 32
        tail = t.tail()
        deg = np.bincount(tail, minlength=t.n_nodes)
        for g in range(n):
            assert all(deg[m.cu(g, c)] == 1 for c in range(128)) and all(deg[m.channel(g, c)] == 1 for c in range(256))
            assert all(deg[m.io(g, p)] == 2 for p in range(32))
            # a corner router: 2 mesh links + 4 CUs + 16 channels + 4 I/O ports
            assert deg[m.router(g, 0, 0)] == 2 + 4 + 16 + 4 and deg[m.router(g, 1, 3)] == 4 + 4
            ch_bw = sum(int(t.bw_q8[t.link_id(m.router(g, *m.channel_router(c)), m.channel(g, c))]) for c in range(256))
            io_bw = sum(int(t.bw_q8[t.link_id(m.io(g, p), m.fabric(p))]) for p in range(32))
            mesh_bw = int(t.bw_q8[t.link_id(m.router(g, 0, 0), m.router(g, 0, 1))])
            assert ch_bw == 4 * mesh_bw and io_bw == mesh_bw
        assert all(deg[m.fabric(p)] == n for p in range(32))


@pytest.mark.parametrize("cu,ch,hops", [(0, 0, 0), (127, 0, 10), (5, 255, 9)])
def test_noc_single_store_closed_form(cu, ch, hops):
    """CF1 over a route with a bottleneck: a store of n lines from one CU to a memory channel of the other GPU.  alpha =
    CU attach 4 + I/O attach 4 + 2 x 1024 scale-up + I/O attach 4 + mesh hops x 4 + channel 64 (all minimum-latency routes
    have the same alpha: `hops` is the Manhattan distance left over after leaving and entering through the nearest side
    column); the channel's 1/8 line per cycle is the bottleneck: t_deliv = 1 + alpha + 8 (n - 1), t_ack = t_deliv + alpha."""
    t, m = noc.noc_cluster(2)
    n = 40
    b = CollectiveBuilder(t.n_gpus, "store")
    b.add(m.cu(0, cu), m.channel(1, ch), n, 0, 1)
    r = oracle.run_workload(_single(t, b.build(), GpuCfg(1, 4, 64, 4)))[0]
    alpha = 4 + 4 + 2048 + 4 + 4 * hops + 64
    assert r.status == 0
    assert r.step_ts.astype(np.int64).tolist() == [[0, 9, 1 + alpha + 8 * (n - 1), 1 + 2 * alpha + 8 * (n - 1)]]


def test_noc_all_gather_conserves_lines():
    t, m = noc.noc_cluster(2)
    ag = noc.noc_all_gather(m, 512, 32, 4)
    assert ag.n_steps == 2 * 32 * 4 * 3 and ag.total_lines == 2 * (512 * 2 + 32 * 4)
    r = oracle.run_workload(_single(t, ag, GpuCfg(1, 4, 64, 4)), flags=oracle.FLAG_PRUNED_SCAN)[0]
    assert r.status == 0
    # every remote store crosses exactly one scale-up switch: lines into the fabric = lines stored remotely
    into_fabric = sum(int(r.link_lines[t.link_id(m.io(g, p), m.fabric(p))]) for g in range(2) for p in range(32))
    assert into_fabric == 2 * 512


@pytest.mark.gpu
def test_noc_engine_parity():
    """Engine vs oracle on a two-GPU NoC cluster (928 nodes, 2,000 links, 4-cycle lookahead window): CU-level all-gather
    with and without the local loads, and a store burst onto one memory channel."""
    from tests.parity import check_workload
    t, m = noc.noc_cluster(2)
    gpu = GpuCfg(1, 4, 64, 4)
    check_workload(_single(t, noc.noc_all_gather(m, 512, 32, 4), gpu), oracle_flags=oracle.FLAG_PRUNED_SCAN)
    check_workload(_single(t, noc.noc_all_gather(m, 300, 8, 2, local_load=False), gpu), oracle_flags=oracle.FLAG_PRUNED_SCAN)
    b = CollectiveBuilder(t.n_gpus, "burst")
    for cu in range(0, 128, 8):
        b.add(m.cu(0, cu), m.channel(1, 3), 20, 0, 1)
    check_workload(_single(t, b.build(), gpu), oracle_flags=oracle.FLAG_PRUNED_SCAN)
    check_workload(_single(t, b.build(), gpu), flags=0x100, oracle_flags=oracle.FLAG_PRUNED_SCAN)


@pytest.mark.gpu
def test_noc_engine_parity_four_gpus():
    """Four NoC-level GPUs (1,824 nodes, 4,000 links, 1,536 endpoints): the CU-level all-gather with local loads, every
    remote store crossing two meshes and one of the 32 scale-up switches."""
    from tests.parity import check_workload
    t, m = noc.noc_cluster(4)
    check_workload(_single(t, noc.noc_all_gather(m, 1024, 32, 4), GpuCfg(1, 4, 64, 4)), oracle_flags=oracle.FLAG_PRUNED_SCAN)
