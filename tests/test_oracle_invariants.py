"""Invariants I1-I9 of SURVEY.md 8(c) as property tests on the oracle, the brute-force
agreement with the independently structured tests/tiny_sim.py, and the equivalence of the
oracle's pruned phase-D scan with its plain scan."""
import numpy as np
import pytest

from astra_inputs import GpuCfg, collectives as C, configs, topologies as T
from oracle import oracle
from tests import tiny_sim


def _route_hops(topo, nl, o, d):
    links, v = [], o
    while v != d:
        e = int(nl[v, d]); links.append(e); v = int(topo.head[e])
        assert len(links) <= topo.n_nodes
    return links


def _check_invariants(topo, coll, gpu, res):
    assert res.status == 0
    S, E = coll.n_steps, topo.n_links
    dist, nl = oracle.route(topo)
    ts = res.step_ts.astype(np.int64)
    # I2: per-link counts equal the lines routed over the link
    expect = np.zeros(E, dtype=np.int64)
    for s in range(S):
        for e in _route_hops(topo, nl, int(coll.owner[s]), int(coll.dst[s])):
            expect[e] += int(coll.lines[s])
    assert res.link_lines.astype(np.int64).tolist() == expect.tolist()
    # I5
    for s in range(S):
        a = int(dist[coll.owner[s], coll.dst[s]])
        rel, iss, dlv, ack = ts[s]
        assert 0 <= rel <= iss
        assert dlv >= iss + 1 + a
        assert ack == dlv + a
        for i in range(int(coll.dep_ptr[s]), int(coll.dep_ptr[s + 1])):
            p, k = int(coll.dep_step[i]), int(coll.dep_kind[i])
            stamp = ts[p][{0: 2, 1: 3, 2: 1}[k]]
            assert rel >= stamp + (1 if k == 2 else 0)      # ISSUED is stamped after phase C
    assert res.completion == ts[:, 3].max()
    # I4 via stats
    assert res.stats[5] <= gpu.max_outstanding and res.stats[4] <= gpu.hbm_lines_per_cycle
    # I9 lower bounds
    sent = np.zeros(topo.n_gpus, dtype=np.int64)
    for s in range(S):
        sent[coll.owner[s]] += int(coll.lines[s])
    for g in range(topo.n_gpus):
        cap = sum(-(-int(topo.bw_q8[e]) // 256) for e in range(int(topo.row_ptr[g]), int(topo.row_ptr[g + 1])))
        if cap:
            assert res.completion >= sent[g] // cap
    if res.trace is not None:
        tr = res.trace.astype(np.int64)
        acc = tr[tr[:, 1] == oracle.TR_ACCEPT]
        # I3: per link per cycle accepted <= ceil(B); over any window of D cycles <= B*D + ceil(B)
        for e in range(E):
            cyc = acc[acc[:, 4] == e][:, 0]
            if cyc.size == 0:
                continue
            bwq = int(topo.bw_q8[e]); ceilb = -(-bwq // 256)
            counts = np.bincount(cyc)
            assert counts.max() <= ceilb
            cum = np.concatenate([[0], np.cumsum(counts)])
            for d in (1, 3, 7, 20):
                if cum.size > d:
                    win = cum[d:] - cum[:-d]
                    assert win.max() * 256 <= bwq * d + ceilb * 256
        iss = tr[tr[:, 1] == oracle.TR_ISSUE]
        # I4: per GPU per cycle issued <= H, one line per wavefront per cycle
        key = iss[:, 0] * 65536 * 4096 + iss[:, 3]
        assert np.unique(key).size == key.size
        gk = iss[:, 0] * 4096 + iss[:, 3] // 65536
        if gk.size:
            assert np.bincount(np.unique(gk, return_inverse=True)[1]).max() <= gpu.hbm_lines_per_cycle
        # conservation: every issued line is accepted hops times, delivered once, acked once
        assert (tr[:, 1] == oracle.TR_DELIVER).sum() == iss.shape[0] == (tr[:, 1] == oracle.TR_ACK).sum()


@pytest.mark.parametrize("seed", range(40))
def test_invariants_random(seed):
    w = configs.random_workload(seed, n_points=2)
    for i in range(w.n_points):
        topo, coll, gpu = w.point(i)
        res = oracle.run_point(topo, coll, gpu, trace_cap=400000)
        _check_invariants(topo, coll, gpu, res)


@pytest.mark.parametrize("seed", range(40))
def test_bruteforce_agreement_random(seed):
    """Oracle (C) == tiny_sim (Python, different structure) on <=4-GPU random cases."""
    w = configs.random_workload(100 + seed, n_points=2, max_lines=40)
    for i in range(w.n_points):
        topo, coll, gpu = w.point(i)
        a = oracle.run_point(topo, coll, gpu)
        b = tiny_sim.simulate(topo, coll, gpu)
        assert a.status == b["status"] == 0
        assert a.completion == b["completion"]
        assert a.step_ts.astype(np.int64).tolist() == b["step_ts"]
        assert a.link_lines.astype(np.int64).tolist() == b["link_lines"]


@pytest.mark.parametrize("mode", [1, 2, 3])
@pytest.mark.parametrize("seed", range(12))
def test_bruteforce_agreement_per_cu_modes(seed, mode):
    """The per-CU readings (R12' one line per CU per cycle, R2' outstanding cap per CU): oracle == tiny_sim on
    random cases, plain and pruned scan alike, and never faster to issue than the per-wavefront reading allows."""
    import dataclasses
    w = configs.random_workload(300 + seed, n_points=2, max_lines=40)
    for i in range(w.n_points):
        topo, coll, gpu0 = w.point(i)
        gpu = dataclasses.replace(gpu0, mode=mode)
        a = oracle.run_point(topo, coll, gpu)
        a2 = oracle.run_point(topo, coll, gpu, flags=oracle.FLAG_PRUNED_SCAN)
        b = tiny_sim.simulate(topo, coll, gpu)
        assert a.status == b["status"] == 0
        assert a.step_ts.astype(np.int64).tolist() == b["step_ts"]
        assert a.link_lines.astype(np.int64).tolist() == b["link_lines"]
        assert (a.step_ts == a2.step_ts).all() and (a.link_lines == a2.link_lines).all()
        assert (a.link_lines == oracle.run_point(topo, coll, gpu0).link_lines).all()      # same routes, same counts


def _small_named_cases():
    cases = []
    gpu = GpuCfg(8, 2, 4, 6)
    cases.append(("ring8", T.ring(8, 256, 9), C.ring_allreduce(8, 203, 8)[0], gpu))
    cases.append(("torus_direct", T.torus2d(2, 4, 128, 7), C.direct_allreduce(8, 170, 8), gpu))
    cases.append(("ring_dbt", T.ring(8, 512, 5), C.double_binary_tree_allreduce(8, 157, 8), gpu))
    cases.append(("torus_hd", T.torus2d(2, 4, 384, 11), C.halving_doubling_allreduce(8, 99, 8), gpu))
    cases.append(("switch_direct", T.single_switch(4, 512, 6, 3), C.direct_allreduce(4, 120, 8), gpu))
    cases.append(("hier", T.nodes_fat_tree(2, 2, 2, 512, 5, 2, 128, 13, 1),
                  C.hierarchical_allreduce(2, 2, 64, 8), gpu))
    r = __import__("astra_inputs").SplitMix64(7)
    cases.append(("a2a_rail", T.rail_optimized(2, 8, 512, 5, 2, 256, 9, 0),
                  C.all_to_all(16, lambda g, d: 1 + (g * 7 + d * 3) % 9, 8), gpu))
    return cases


@pytest.mark.parametrize("case", _small_named_cases(), ids=lambda c: c[0])
def test_invariants_and_bruteforce_named_families(case):
    """Every collective family on a small instance of its topology family."""
    _, topo, coll, gpu = case
    res = oracle.run_point(topo, coll, gpu, trace_cap=2000000)
    _check_invariants(topo, coll, gpu, res)
    b = tiny_sim.simulate(topo, coll, gpu)
    assert res.step_ts.astype(np.int64).tolist() == b["step_ts"]
    assert res.link_lines.astype(np.int64).tolist() == b["link_lines"]


def test_i6_determinism():
    w = configs.random_workload(5, n_points=3)
    a = oracle.run_workload(w)
    b = oracle.run_workload(w, processes=2)
    for x, y in zip(a, b):
        assert x.completion == y.completion and (x.step_ts == y.step_ts).all() and (x.link_lines == y.link_lines).all()


@pytest.mark.parametrize("family", ["ring", "torus_direct"])
def test_i7_completion_non_increasing_in_bandwidth(family):
    prev = None
    for bw in (64, 128, 256, 512, 1024, 2048):
        if family == "ring":
            topo, coll = T.ring(8, bw, 40), C.ring_allreduce(8, 640, 8)[0]
        else:
            topo, coll = T.torus2d(2, 4, bw, 40), C.direct_allreduce(8, 640, 8)
        r = oracle.run_point(topo, coll, GpuCfg(8, 2, 8, 8))
        assert prev is None or r.completion <= prev
        prev = r.completion


@pytest.mark.parametrize("seed", range(25))
def test_pruned_scan_equals_plain_scan_random(seed):
    w = configs.random_workload(300 + seed, n_points=2, max_gpus=6, max_steps=30, max_lines=300)
    for i in range(w.n_points):
        topo, coll, gpu = w.point(i)
        a = oracle.run_point(topo, coll, gpu)
        b = oracle.run_point(topo, coll, gpu, flags=oracle.FLAG_PRUNED_SCAN)
        assert a.status == b.status == 0 and a.completion == b.completion
        assert (a.step_ts == b.step_ts).all() and (a.link_lines == b.link_lines).all()
        assert b.stats[6] <= a.stats[6]


def test_pruned_scan_equals_plain_scan_configs():
    w1 = configs.config1()
    w2 = configs.config2(range(6, 10))
    w4 = configs.config4(12).subset([1, 3, 5, 6, 8, 9, 11])   # the cheap ones (< 35k cycles each)
    for w in (w1, w2, w4):
        a = oracle.run_workload(w)
        b = oracle.run_workload(w, flags=oracle.FLAG_PRUNED_SCAN)
        for x, y in zip(a, b):
            assert x.status == y.status == 0
            assert x.completion == y.completion and (x.step_ts == y.step_ts).all() and (x.link_lines == y.link_lines).all()


def test_watchdog_status():
    topo, coll, gpu = configs.config1().point(0)
    r = oracle.run_point(topo, coll, gpu, max_cycles=1000)
    assert r.status == 1


def test_validation_errors():
    topo, coll, gpu = configs.config1().point(0)
    bad = GpuCfg(2, 2, 16, 8)           # CU range [0,4) exceeds 2 CUs
    r = oracle.run_point(topo, coll, bad, check=False)
    assert r.status == -1
    line3 = T.Topology.from_edges(3, 0, [0, 0, 0], [(0, 1, 256, 5), (1, 0, 256, 5)])
    r = oracle.run_point(line3, C.single_transfer(3, 0, 2, 4, 0, 1), GpuCfg(1, 1, 4, 1), check=False)
    assert r.status == -4               # unreachable
