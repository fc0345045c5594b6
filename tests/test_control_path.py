"""Control-path variants of a step DAG (second slice): put + signal
(SemaphoreRelease as a one-line transaction from wavefront zero behind a step)
and get (request -> response) as transforms of the collective, run through the unchanged
oracle and engine.  Expected values: tests/golden/pins_control_path.json (hand traces, closed form)."""
import json
import os

import numpy as np
import pytest

from astra_inputs import GpuCfg, Workload, collectives as C, configs, topologies as T
from astra_inputs.types import CollectiveBuilder, DEP_ACKED, DEP_DELIVERED, DEP_ISSUED
from oracle import oracle

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "pins_control_path.json")))


def _single(topo, coll, gpu, max_cycles=1 << 30):
    w = Workload(name=coll.name or "case", max_cycles=max_cycles)
    w.topologies.append(topo); w.collectives.append(coll); w.gpus.append(gpu)
    w.points.append((0, 0, 0)); w.meta.append({})
    return w


def _two_step_case():
    topo = T.Topology.from_edges(2, 0, [0, 0], [(0, 1, 256, 3), (1, 0, 256, 3)])
    b = CollectiveBuilder(2, "two_steps")
    a = b.add(0, 1, 5, 0, 1)
    b.add(1, 0, 1, 0, 1, [(a, DEP_DELIVERED)])
    return topo, b.build(), GpuCfg(1, 1, 64, 1)


def _barrier_cases():
    """(key in the golden file, variant name, topology, collective, GPU) of the NopOp / BarrierOp / fence hand traces."""
    topo = T.Topology.from_edges(2, 0, [0, 0], [(0, 1, 1024, 3), (1, 0, 1024, 3)])
    b = CollectiveBuilder(2, "ab"); b.add(0, 1, 5, 0, 1); b.add(0, 1, 4, 0, 1)
    ab, g1 = b.build(), GpuCfg(1, 2, 64, 2)
    b = CollectiveBuilder(2, "xyz"); b.add(0, 1, 4, 0, 1); b.add(0, 1, 2, 1, 1); b.add(0, 1, 2, 1, 1)
    xyz, g2 = b.build(), GpuCfg(2, 1, 64, 2)
    return [("S4_nop_and_fence", "plain", topo, ab, g1),
            ("S4_nop_and_fence", "nop", topo, C.with_barriers(ab, 1, "workgroup", DEP_ISSUED), g1),
            ("S4_nop_and_fence", "fence", topo, C.with_barriers(ab, 1, "workgroup", DEP_ACKED), g1),
            ("S5_barrier_scope", "plain", topo, xyz, g2),
            ("S5_barrier_scope", "workgroup", topo, C.with_barriers(xyz, 2, "workgroup", DEP_ISSUED), g2),
            ("S5_barrier_scope", "gpu", topo, C.with_barriers(xyz, 2, "gpu", DEP_ISSUED), g2)]


def _transformed_workloads():
    """Small workloads for engine-vs-oracle parity: every named family with both transforms."""
    out = []
    topo, coll, gpu = configs.config1().point(0)
    out += [_single(topo, C.put_with_signal(coll), gpu), _single(topo, C.as_get(coll), gpu), _single(topo, C.as_get(coll, 300), gpu)]
    w2 = configs.config2(range(6, 8))
    for i in range(w2.n_points):
        t2, c2, g2 = w2.point(i)
        out += [_single(t2, C.put_with_signal(c2), g2), _single(t2, C.as_get(c2, 64), g2)]
    w4 = configs.config4(6)
    for i in range(w4.n_points):
        t4, c4, g4 = w4.point(i)
        out += [_single(t4, C.put_with_signal(c4), g4), _single(t4, C.as_get(c4), g4)]
    out += [_single(topo, C.with_barriers(coll, gpu.cus, "workgroup", DEP_ISSUED), gpu), _single(topo, C.with_barriers(coll, gpu.cus, "gpu", DEP_ACKED), gpu)]
    t2, c2, g2 = w2.point(1)
    out += [_single(t2, C.with_barriers(c2, g2.cus, "workgroup", DEP_ACKED), g2), _single(t2, C.with_barriers(c2, g2.cus, "gpu", DEP_ISSUED), g2)]
    for seed in (3, 4, 5):
        wr = configs.random_workload(seed, n_points=2, max_gpus=6, max_steps=16, max_lines=120)
        for i in range(wr.n_points):
            tr, cr, gr = wr.point(i)
            if all(int(k) == DEP_DELIVERED for k in cr.dep_kind):       # as_get keeps kinds; signals need DELIVERED waits
                out.append(_single(tr, C.as_get(cr, 40), gr))
            out.append(_single(tr, C.put_with_signal(cr), gr))
    return out


# ---------------------------------------------------------------------------------------------
# the transforms themselves (inputs): structure
# ---------------------------------------------------------------------------------------------
def test_put_with_signal_structure():
    for w in (configs.config1(), configs.config2(range(6, 7))):
        for i in range(w.n_points):
            _, coll, gpu = w.point(i)
            sig = C.put_with_signal(coll)
            waited = {int(p) for p, k in zip(coll.dep_step, coll.dep_kind) if int(k) == DEP_DELIVERED}
            assert sig.n_steps == coll.n_steps + len(waited)
            assert sig.total_lines == coll.total_lines + len(waited)
            n_sig = 0
            for s in range(sig.n_steps):
                deps = [(int(sig.dep_step[j]), int(sig.dep_kind[j])) for j in range(int(sig.dep_ptr[s]), int(sig.dep_ptr[s + 1]))]
                if deps and deps[0][1] == DEP_ISSUED:                 # a signal: one line, one CU, right behind its step
                    n_sig += 1
                    p = deps[0][0]
                    assert p == s - 1 and int(sig.lines[s]) == 1 and int(sig.cu_n[s]) == 1
                    assert int(sig.owner[s]) == int(sig.owner[p]) and int(sig.dst[s]) == int(sig.dst[p]) and int(sig.cu_lo[s]) == int(sig.cu_lo[p])
                for p, k in deps:
                    if k == DEP_DELIVERED:                            # data steps wait for signals only
                        assert int(sig.lines[p]) == 1 and int(sig.dst[p]) == int(sig.owner[s])
            assert n_sig == len(waited)


def test_as_get_structure():
    _, coll, _ = configs.config2(range(6, 7)).point(1)
    for chunk in (0, 16, 1000):
        g = C.as_get(coll, chunk)
        req = [s for s in range(g.n_steps) if int(g.dep_ptr[s + 1]) == int(g.dep_ptr[s]) and int(g.lines[s]) == 1]
        resp = [s for s in range(g.n_steps) if s not in set(req)]
        assert len(req) == len(resp)
        assert sum(int(g.lines[s]) for s in resp) == coll.total_lines
        for s in resp:                                                # the request right before it, in the other direction
            assert int(g.owner[s - 1]) == int(g.dst[s]) and int(g.dst[s - 1]) == int(g.owner[s])
            deps = [(int(g.dep_step[j]), int(g.dep_kind[j])) for j in range(int(g.dep_ptr[s]), int(g.dep_ptr[s + 1]))]
            assert (s - 1, DEP_DELIVERED) in deps


# ---------------------------------------------------------------------------------------------
# oracle against the hand traces and the closed form
# ---------------------------------------------------------------------------------------------
def test_signal_hand_trace():
    topo, coll, gpu = _two_step_case()
    r = oracle.run_workload(_single(topo, C.put_with_signal(coll), gpu))[0]
    g = GOLD["S1_put_signal"]
    assert r.status == 0 and r.completion == g["completion"]
    assert r.step_ts.astype(np.int64).tolist() == g["step_ts"]
    assert oracle.run_workload(_single(topo, coll, gpu))[0].completion == g["put_completion"]


def test_get_hand_trace():
    topo, coll, gpu = _two_step_case()
    r = oracle.run_workload(_single(topo, C.as_get(coll), gpu))[0]
    g = GOLD["S2_get"]
    assert r.status == 0 and r.completion == g["completion"]
    assert r.step_ts.astype(np.int64).tolist() == g["step_ts"]


def test_barrier_hand_traces():
    """NopOp (ISSUED), fence (ACKED) and BarrierOp (GPU scope) as dependencies between a GPU's own steps."""
    for key, name, topo, coll, gpu in _barrier_cases():
        r = oracle.run_workload(_single(topo, coll, gpu))[0]
        assert r.status == 0 and r.step_ts.astype(np.int64).tolist() == GOLD[key][name], (key, name)


def test_ring_signal_closed_form():
    """T = 14 (350 + n/4) + 13 + 350: one more accept slot per signalled ring step (derivation in the golden file)."""
    w2 = configs.config2(range(6, 10))
    for i in range(w2.n_points):
        if w2.meta[i]["algo"] != "ring":
            continue
        topo, coll, gpu = w2.point(i)
        n = w2.meta[i]["lines"] // 8
        r = oracle.run_workload(_single(topo, C.put_with_signal(coll), gpu))[0]
        assert r.status == 0
        assert r.completion == 14 * (350 + n // 4) + 13 + 350 == GOLD["S3_ring_signal_config2"]["completion"][str(w2.meta[i]["lines"])]


def test_control_variants_keep_the_invariants():
    """I2 (lines per link = lines routed over it), I5 (release <= issued, ack = deliv + alpha) on the transformed DAGs,
    and: a signal can only delay the steps that wait for it."""
    for w in _transformed_workloads()[:9]:
        r = oracle.run_workload(w)[0]
        assert r.status == 0
        ts = r.step_ts.astype(np.int64)
        assert (ts[:, 0] <= ts[:, 1]).all() and (ts[:, 1] < ts[:, 2]).all() and (ts[:, 2] < ts[:, 3]).all()
        assert int(r.link_lines.sum()) >= int(w.collectives[0].total_lines)
    topo, coll, gpu = configs.config1().point(0)
    assert oracle.run_workload(_single(topo, C.put_with_signal(coll), gpu))[0].completion >= 38623


# ---------------------------------------------------------------------------------------------
# engine against the oracle
# ---------------------------------------------------------------------------------------------
@pytest.mark.gpu
def test_engine_matches_hand_traces():
    from paper_2606_10440_b200 import simulate_workload
    topo, coll, gpu = _two_step_case()
    for key, cc in (("S1_put_signal", C.put_with_signal(coll)), ("S2_get", C.as_get(coll))):
        summ, ts, _ = simulate_workload(_single(topo, cc, gpu))[0]
        assert summ.status == 0 and summ.completion_cycle == GOLD[key]["completion"]
        assert ts.astype(np.int64).tolist() == GOLD[key]["step_ts"]
    for key, name, topo, cc, gpu in _barrier_cases():
        summ, ts, _ = simulate_workload(_single(topo, cc, gpu))[0]
        assert summ.status == 0 and ts.astype(np.int64).tolist() == GOLD[key][name], (key, name)


@pytest.mark.gpu
def test_engine_parity_on_control_variants():
    from tests.parity import check_workload
    for w in _transformed_workloads():
        check_workload(w, oracle_flags=oracle.FLAG_PRUNED_SCAN)
        check_workload(w, flags=0x100, oracle_flags=oracle.FLAG_PRUNED_SCAN)       # one CTA per point


@pytest.mark.gpu
def test_engine_ring_signal_closed_form_all_sizes():
    """Config 2's ring with signals at all eleven sizes (64 KiB .. 64 MiB) on the engine: T = 14 (350 + n/4) + 13 + 350
    (the closed form the oracle is pinned to at the four smallest sizes, derivation in the golden file)."""
    from paper_2606_10440_b200 import simulate_workload
    w2 = configs.config2()
    ws = Workload(name="ring+signal", max_cycles=w2.max_cycles)
    expect = []
    for i in range(w2.n_points):
        if w2.meta[i]["algo"] != "ring":
            continue
        topo, coll, gpu = w2.point(i)
        ws.topologies.append(topo); ws.collectives.append(C.put_with_signal(coll)); ws.gpus.append(gpu)
        ws.points.append((len(ws.topologies) - 1, len(ws.collectives) - 1, len(ws.gpus) - 1)); ws.meta.append({})
        expect.append(14 * (350 + w2.meta[i]["lines"] // 8 // 4) + 13 + 350)
    res = simulate_workload(ws)
    assert len(res) == 11
    for (summ, _, _), t in zip(res, expect):
        assert summ.status == 0 and summ.completion_cycle == t
