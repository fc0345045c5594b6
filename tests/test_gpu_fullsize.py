"""BASELINE configs 3, 4 (all 4,096 points) and 5 at FULL size through the CUDA engine in the launch
configuration bench.py uses (engine's choice of CTA groups), compared with the CPU oracle for EVERY
design point: status, completion cycle, total lines and the SHA-256 of the [S,4] step-timestamp array
and of the per-link line counts, against tests/golden/full_size.json.  That file is written by
tests/golden/make_full_size.py from `oracle/` and `astra_inputs/` only (the oracle needs minutes to
hours at these sizes, so it is run once and its digests are stored); no value in it comes from the
CUDA path.  A mismatch is a finding about the engine, never a reason to touch the golden file.
On top of that the invariants that hold at any size are checked on the arrays themselves: I2
(per-link counts == lines routed over the link, routes from the oracle's own router), I5 (release <=
issued, delivered >= issued + 1 + alpha, acked == delivered + alpha exactly, every dependency
honoured), R10, I9 lower bounds, completion == max t_ack."""
import hashlib
import json
import os

import numpy as np
import pytest

from astra_inputs import configs
from oracle import oracle
from tests.parity import compare_point

pytestmark = pytest.mark.gpu

_GOLD_PATH = os.path.join(os.path.dirname(__file__), "golden", "full_size.json")
GOLD = json.load(open(_GOLD_PATH)) if os.path.exists(_GOLD_PATH) else {}


def _digest(arr):
    return hashlib.sha256(np.ascontiguousarray(arr, dtype="<u8").tobytes()).hexdigest()


def _check_golden(cfg_key, i, res):
    """Engine result of design point i == the oracle's stored digests."""
    summ, ts, ll = res
    assert cfg_key in GOLD and str(i) in GOLD[cfg_key], f"{cfg_key}[{i}] missing from tests/golden/full_size.json"
    status, completion, total, h_ts, h_ll, _scan = GOLD[cfg_key][str(i)]
    label = f"{cfg_key}[{i}]"
    assert summ.status == status, f"{label}: status {summ.status} != oracle {status}"
    assert summ.completion_cycle == completion, f"{label}: completion {summ.completion_cycle} != oracle {completion}"
    assert summ.total_lines == total, label
    assert _digest(ll) == h_ll, f"{label}: link_lines differ from the oracle's"
    assert _digest(ts) == h_ts, f"{label}: step timestamps differ from the oracle's"


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


def test_config3_full_size_vs_oracle():
    from paper_2606_10440_b200 import simulate_workload
    w = configs.config3()
    res = simulate_workload(w)
    topo, coll, _ = w.point(0)
    assert res[0][0].total_lines == 264241152
    _check_golden("config3", 0, res[0])
    _check_point(topo, coll, res[0])


def test_config5_full_size_vs_oracle():
    from paper_2606_10440_b200 import simulate_workload
    w = configs.config5()
    res = simulate_workload(w)
    topo, coll, _ = w.point(0)
    _check_golden("config5", 0, res[0])
    _check_point(topo, coll, res[0])


def test_config4_all_4096_points_vs_oracle():
    """One batch of all 4,096 points, exactly what bench.py times; every point against the oracle's digests."""
    from paper_2606_10440_b200 import simulate_workload
    w = configs.config4()
    res = simulate_workload(w)
    assert len(res) == 4096
    bad = []
    for i in range(w.n_points):
        try:
            _check_golden("config4", i, res[i])
        except AssertionError as e:
            bad.append(str(e))
    assert not bad, f"{len(bad)} of 4096 points differ from the oracle; first: {bad[:3]}"
    for i in range(0, w.n_points, 8):                      # invariants on a 512-point stride
        topo, coll, _ = w.point(i)
        _check_point(topo, coll, res[i])
