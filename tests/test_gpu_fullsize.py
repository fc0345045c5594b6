"""BASELINE configs 3, 4 (a 512-point slice) and 5 at FULL size through the CUDA engine in the launch
configuration bench.py uses (engine's choice of CTA group).  The oracle needs minutes per point at
these sizes, so what is checked here holds at any size: I2 (per-link counts == lines routed over
the link, routes from the oracle's own router), I5 (release <= issued, delivered >= issued + 1 +
alpha, acked == delivered + alpha exactly, every dependency honoured), I9 lower bounds, completion
== max t_ack -- plus, for config 4, sampled points compared bit for bit with the oracle."""
import numpy as np
import pytest

from astra_inputs import configs
from oracle import oracle
from tests.parity import compare_point

pytestmark = pytest.mark.gpu


def _check_point(topo, coll, res):
    summ, ts, ll = res
    assert summ.status == 0
    dist, nl = oracle.route(topo)
    S, E = coll.n_steps, topo.n_links
    owner, dst, lines = coll.owner.astype(np.int64), coll.dst.astype(np.int64), coll.lines.astype(np.int64)
    # I2 -- routes walked once per (owner, dst) pair
    expect = np.zeros(E, dtype=np.int64)
    pair_lines = {}
    for s in range(S):
        pair_lines[(int(owner[s]), int(dst[s]))] = pair_lines.get((int(owner[s]), int(dst[s])), 0) + int(lines[s])
    head = topo.head
    for (o, d), n in pair_lines.items():
        v, hops = o, 0
        while v != d:
            e = int(nl[v, d]); expect[e] += n; v = int(head[e]); hops += 1
            assert hops <= topo.n_nodes
    assert (ll.astype(np.int64) == expect).all()
    # I5
    t = ts.astype(np.int64)
    alpha = dist[owner, dst].astype(np.int64)
    assert (t[:, 0] >= 0).all() and (t[:, 0] <= t[:, 1]).all()
    assert (t[:, 2] >= t[:, 1] + 1 + alpha).all()
    assert (t[:, 3] == t[:, 2] + alpha).all()
    dep_ptr, dep_step, dep_kind = coll.dep_ptr.astype(np.int64), coll.dep_step.astype(np.int64), coll.dep_kind.astype(np.int64)
    cons = np.repeat(np.arange(S), np.diff(dep_ptr))
    col = np.array([2, 3, 1])[dep_kind]
    stamp = t[dep_step, col] + (dep_kind == 2)
    assert (t[cons, 0] >= stamp).all()
    # R10: a step is released exactly when its last dependency is satisfied
    last = np.zeros(S, dtype=np.int64)
    np.maximum.at(last, cons, stamp)
    assert (t[:, 0] == last).all()
    assert summ.completion_cycle == t[:, 3].max()
    # I9
    sent = np.bincount(owner, weights=lines, minlength=topo.n_gpus)
    for g in range(topo.n_gpus):
        cap = sum(-(-int(topo.bw_q8[e]) // 256) for e in range(int(topo.row_ptr[g]), int(topo.row_ptr[g + 1])))
        if cap:
            assert summ.completion_cycle >= sent[g] // cap


def test_config3_full_size_invariants():
    from paper_2606_10440_b200 import simulate_workload
    w = configs.config3()
    res = simulate_workload(w)
    topo, coll, _ = w.point(0)
    assert res[0][0].total_lines == 264241152
    _check_point(topo, coll, res[0])


def test_config5_full_size_invariants():
    from paper_2606_10440_b200 import simulate_workload
    w = configs.config5()
    res = simulate_workload(w)
    topo, coll, _ = w.point(0)
    _check_point(topo, coll, res[0])


def test_config4_slice_invariants_and_sampled_parity():
    from paper_2606_10440_b200 import simulate_workload
    w = configs.config4(512)
    res = simulate_workload(w)
    for i in range(w.n_points):
        topo, coll, _ = w.point(i)
        _check_point(topo, coll, res[i])
    cheap = sorted(range(w.n_points), key=lambda i: w.collectives[w.points[i][1]].total_lines)[:48]
    sample = cheap[::4] + [cheap[-1]]
    ora = oracle.run_workload(w, sample, processes=8, flags=oracle.FLAG_PRUNED_SCAN)
    for j, i in enumerate(sample):
        compare_point(res[i], ora[j], label=f"config4[{i}]")
