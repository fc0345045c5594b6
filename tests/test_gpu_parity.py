"""Parity proper: CUDA engine (through the C-ABI) == CPU oracle, bit for bit, on every integer
output (completion cycle, four timestamps per step, lines per link).  Needs a B200."""
import os

import numpy as np
import pytest

from astra_inputs import GpuCfg, Workload, collectives as C, configs, topologies as T
from oracle import oracle
from tests.parity import check_workload, compare_point

pytestmark = pytest.mark.gpu

FLAG_NO_WINDOW_SKIP, FLAG_WINDOW_1, FLAG_SERIAL_ISSUE, FLAG_SERIAL_ARRIVALS, FLAG_NO_HEAVY, FLAG_NO_PRIORITY_SWEEP = 1, 2, 4, 8, 16, 32
FLAG_RUN_AHEAD = 64


def _single(topo, coll, gpu, name="case", max_cycles=1 << 22):
    w = Workload(name=name, max_cycles=max_cycles)
    w.topologies.append(topo); w.collectives.append(coll); w.gpus.append(gpu)
    w.points.append((0, 0, 0)); w.meta.append({})
    return w


def test_library_loaded_is_in_tree():
    import paper_2606_10440_b200 as pkg
    lib = pkg.load_library()
    assert os.path.dirname(lib._name) == os.path.dirname(pkg.__file__)


@pytest.mark.parametrize("k", [64, 2])
def test_p1_hand_trace(k):
    check_workload(_single(T.line(2, 256, 3), C.single_transfer(2, 0, 1, 5, 0, 1), GpuCfg(1, 1, k, 1)))


def test_p2_p3():
    check_workload(_single(T.line(2, 128, 3), C.single_transfer(2, 0, 1, 5, 0, 1), GpuCfg(1, 2, 64, 2)))
    check_workload(_single(T.line(2, 1024, 7), C.single_transfer(2, 0, 1, 10, 0, 2), GpuCfg(2, 4, 64, 8)))


@pytest.mark.parametrize("key", __import__("tests.pin_cases", fromlist=["ROUND2"]).ROUND2)
def test_round2_hand_traces(key):
    """Grant order when H binds, general-credit bandwidths, ISSUED/ACKED release timing: the engine
    against the oracle AND against the hand-derived values of the golden file."""
    from tests import pin_cases
    topo, coll, gpu = pin_cases.build(key)
    res, _ = check_workload(_single(topo, coll, gpu, name=key))
    g = pin_cases.GOLD[key]
    want = g["step_ts"] if isinstance(g["step_ts"][0], list) else [g["step_ts"]]
    assert res[0][1].tolist() == want


@pytest.mark.parametrize("key", __import__("tests.pin_cases", fromlist=["PER_CU"]).PER_CU)
def test_per_cu_hand_traces(key):
    """The paper's per-CU readings (astra_set_gpu_ex: one line per CU per cycle, outstanding cap per CU):
    engine == oracle == the hand-derived values."""
    from tests import pin_cases
    topo, coll, gpu = pin_cases.build(key)
    res, _ = check_workload(_single(topo, coll, gpu, name=key))
    assert res[0][1].tolist() == [pin_cases.GOLD[key]["step_ts"]]


@pytest.mark.parametrize("mode", [1, 2, 3])
def test_per_cu_modes_random_and_families(mode):
    """Per-CU modes on random workloads (all dep kinds, 1-cycle windows), on config 1 and on small instances of
    the collective families, one CTA and CTA groups."""
    import dataclasses
    from paper_2606_10440_b200.binding import FLAG_GROUP
    for seed in (41, 42, 43, 44):
        w = configs.random_workload(seed, n_points=6, max_gpus=6, max_steps=24, max_lines=200)
        w.gpus = [dataclasses.replace(g, mode=mode) for g in w.gpus]
        check_workload(w)
        check_workload(w, flags=FLAG_GROUP(3))
    w = configs.config1()
    w.gpus = [dataclasses.replace(g, mode=mode) for g in w.gpus]
    check_workload(w)
    gpu = GpuCfg(8, 4, 6, 5, mode)
    for topo, coll in [(T.ring(8, 256, 9), C.ring_allreduce(8, 403, 8)[0]),
                       (T.torus2d(2, 4, 128, 7), C.direct_allreduce(8, 370, 8)),
                       (T.single_switch(4, 512, 6, 3), C.direct_allreduce(4, 320, 8)),
                       (T.rail_optimized(2, 8, 512, 5, 2, 256, 9, 0), C.all_to_all(16, lambda g, d: 1 + (g * 7 + d * 3) % 19, 8))]:
        check_workload(_single(topo, coll, gpu))
    w = configs.config2(range(6, 8))
    w.gpus = [dataclasses.replace(g, mode=mode) for g in w.gpus]
    check_workload(w, processes=4)


def test_config1_bit_exact_and_pin():
    gpu, _ = check_workload(configs.config1())
    assert gpu[0][0].completion_cycle == 38623


@pytest.mark.parametrize("cus", [1, 2, 8, 16, 64])
def test_config1_cu_sweep(cus):
    check_workload(configs.config1(cus))


@pytest.mark.parametrize("seed", range(30))
def test_random_small_workloads(seed):
    """Random topologies (latencies down to 1 cycle -> 1-cycle windows), all three dep kinds."""
    check_workload(configs.random_workload(seed, n_points=4, max_gpus=6, max_steps=24, max_lines=200))


@pytest.mark.parametrize("flags", [FLAG_NO_WINDOW_SKIP, FLAG_WINDOW_1, FLAG_NO_WINDOW_SKIP | FLAG_WINDOW_1,
                                   FLAG_RUN_AHEAD | FLAG_WINDOW_1 | 0x100, FLAG_RUN_AHEAD | FLAG_NO_WINDOW_SKIP | FLAG_WINDOW_1 | 0x100])
def test_i8_skip_equivalence(flags):
    """I8: outputs with idle-cycle / window skipping == without, and with a 1-cycle window."""
    w = configs.random_workload(77, n_points=6, max_gpus=6, max_steps=24, max_lines=200)
    check_workload(w, flags=flags)
    check_workload(configs.config1(), flags=flags)


@pytest.mark.parametrize("flags", [FLAG_SERIAL_ISSUE, FLAG_SERIAL_ARRIVALS, FLAG_NO_HEAVY, FLAG_NO_PRIORITY_SWEEP, FLAG_SERIAL_ISSUE | FLAG_SERIAL_ARRIVALS | 0x100,
                                   FLAG_RUN_AHEAD, FLAG_RUN_AHEAD | 0x100, FLAG_RUN_AHEAD | FLAG_NO_WINDOW_SKIP | 0x100])
def test_engine_paths_agree(flags):
    """The wavefront-parallel issue stage and the chunked arrival stage (defaults) and the cycle-serial /
    one-task-per-link paths they fall back to give the same bits; 0x100 = one CTA per point; RUN_AHEAD = no block
    barrier per window, nodes run ahead of the nodes they do not depend on."""
    check_workload(configs.random_workload(91, n_points=6, max_gpus=6, max_steps=24, max_lines=200), flags=flags)
    check_workload(configs.config1(), flags=flags)
    check_workload(configs.config2(range(6, 8)), flags=flags, processes=4)
    check_workload(configs.config4(12), flags=flags, oracle_flags=oracle.FLAG_PRUNED_SCAN, processes=6)


@pytest.mark.parametrize("group", [1, 2, 3, 8])
def test_cta_groups(group):
    """A design point spread over a group of CTAs (one node range each, one group barrier per
    window) gives the same bits as on one CTA."""
    from paper_2606_10440_b200.binding import FLAG_GROUP
    check_workload(configs.config1(), flags=FLAG_GROUP(group))
    check_workload(configs.random_workload(5, n_points=6, max_gpus=6, max_steps=24, max_lines=200), flags=FLAG_GROUP(group))
    check_workload(configs.config2(range(6, 9)), flags=FLAG_GROUP(group), processes=6)
    check_workload(configs.config5(n_nodes=4), flags=FLAG_GROUP(group), oracle_flags=oracle.FLAG_PRUNED_SCAN)


@pytest.mark.parametrize("warps", [1, 2, 4, 8])
def test_warp_sets(warps):
    """CTAs of fewer warps (ASTRA_FLAG_WARPS): a warp set then steps several simulated nodes one after the other,
    or a node gets a set of 1, 2, 4, 8 warps -- every split of a CTA's warps over its nodes gives the same bits."""
    from paper_2606_10440_b200.binding import FLAG_GROUP, FLAG_WARPS
    check_workload(configs.config1(), flags=FLAG_WARPS(warps))
    check_workload(configs.random_workload(23, n_points=6, max_gpus=6, max_steps=24, max_lines=200), flags=FLAG_WARPS(warps))
    check_workload(configs.config2(range(6, 8)), flags=FLAG_WARPS(warps) | FLAG_GROUP(1), processes=4)
    check_workload(configs.config4(8), flags=FLAG_WARPS(warps), oracle_flags=oracle.FLAG_PRUNED_SCAN, processes=8)
    check_workload(configs.config5(n_nodes=4), flags=FLAG_WARPS(warps) | FLAG_GROUP(3), oracle_flags=oracle.FLAG_PRUNED_SCAN)


def test_two_contexts_run_concurrently():
    """Two astra_ctx on the same device, each with its own stream, both launched before either is waited for:
    the cooperative launches are serialised or co-scheduled by the runtime, never deadlocked, and both give the
    oracle's bits."""
    from paper_2606_10440_b200 import Engine
    wa = configs.config2(range(6, 12))
    wb = configs.config5(n_nodes=4)
    with Engine() as ea, Engine() as eb:
        pa, pb = ea.load_workload(wa), eb.load_workload(wb)
        ea.run_batch(pa, wa.max_cycles, asynchronous=True)
        eb.run_batch(pb, wb.max_cycles, asynchronous=True)
        ea.sync(); eb.sync()
        ra = [ea.read_results(i) for i in range(len(pa))]
        rb = [eb.read_results(i) for i in range(len(pb))]
    for i, r in enumerate(oracle.run_workload(wa, processes=6)):
        compare_point(ra[i], r, label=f"ctx A point {i}")
    compare_point(rb[0], oracle.run_workload(wb, flags=oracle.FLAG_PRUNED_SCAN)[0], label="ctx B")


def test_named_families_small():
    gpu = GpuCfg(8, 2, 4, 6)
    cases = [
        (T.ring(8, 256, 9), C.ring_allreduce(8, 203, 8)[0]),
        (T.torus2d(2, 4, 128, 7), C.direct_allreduce(8, 170, 8)),
        (T.ring(8, 512, 5), C.double_binary_tree_allreduce(8, 157, 8)),
        (T.torus2d(2, 4, 384, 11), C.halving_doubling_allreduce(8, 99, 8)),
        (T.single_switch(4, 512, 6, 3), C.direct_allreduce(4, 120, 8)),
        (T.nodes_fat_tree(2, 2, 2, 512, 5, 2, 128, 13, 1), C.hierarchical_allreduce(2, 2, 64, 8)),
        (T.rail_optimized(2, 8, 512, 5, 2, 256, 9, 0), C.all_to_all(16, lambda g, d: 1 + (g * 7 + d * 3) % 9, 8)),
    ]
    for i, (topo, coll) in enumerate(cases):
        check_workload(_single(topo, coll, gpu, name=f"family{i}"))


def test_config2_all_22_points():
    """BASELINE config 2 in the launch configuration bench.py times (one batch of 22 points)."""
    gpu, _ = check_workload(configs.config2(), processes=8)
    w = configs.config2()
    for (summ, _, _), m in zip(gpu, w.meta):
        n = m["lines"] // 8
        if m["algo"] == "ring":
            assert summ.completion_cycle == 14 * (350 + -(-n // 4)) + 350


def test_config3_reduced():
    """Config 3 topology and collective at 1/8 of the message size (33 M lines; oracle finishes in seconds)."""
    check_workload(configs.config3(lines=32 * 1024 * 8))


def test_config5_reduced():
    check_workload(configs.config5(n_nodes=4), oracle_flags=oracle.FLAG_PRUNED_SCAN)


def test_config5_eight_nodes():
    """A quarter of config 5's nodes (64 GPUs, 8 node and 8 rail switches): the engine spreads it over 80 CTAs."""
    check_workload(configs.config5(n_nodes=8), oracle_flags=oracle.FLAG_PRUNED_SCAN)


def test_config4_sample():
    """64 of the 4096 config-4 points (every point is independent): pruned-scan oracle."""
    w = configs.config4(64)
    check_workload(w, oracle_flags=oracle.FLAG_PRUNED_SCAN, processes=8)


def test_i6_batch_independence():
    """A point's result does not depend on its neighbours or on the batch order."""
    from paper_2606_10440_b200 import simulate_workload
    w = configs.config4(24)
    a = simulate_workload(w)
    order = list(reversed(range(24)))
    b = simulate_workload(w, indices=order)
    c = simulate_workload(w, indices=[5])
    for j, i in enumerate(order):
        assert a[i][0].completion_cycle == b[j][0].completion_cycle
        assert (a[i][1] == b[j][1]).all() and (a[i][2] == b[j][2]).all()
    assert (a[5][1] == c[0][1]).all()


@pytest.mark.parametrize("flags", [0, 0x100, FLAG_RUN_AHEAD | 0x100])
def test_watchdog_cuts(flags):
    """Runs cut by max_cycles at many points of the run (inside a window, at a window edge, at the completion cycle
    and one before): status and every timestamp stamped before the cut equal the oracle's, with nodes running ahead
    (one CTA per point, 0x100) and with the barrier per window."""
    topo, coll, gpu = configs.config1().point(0)
    for mc in (0, 1, 191, 192, 193, 5000, 38400, 38592, 38622, 38623, 38624, 38700):
        check_workload(_single(topo, coll, gpu, max_cycles=mc), flags=flags)
    w = configs.random_workload(12, n_points=1, max_gpus=6, max_steps=24, max_lines=200)
    t2, c2, g2 = w.point(0)
    full = check_workload(w, flags=flags)[0][0][0].completion_cycle
    for mc in (full - 1, full, full + 1, full // 2, 7):
        check_workload(_single(t2, c2, g2, max_cycles=max(0, mc)), flags=flags)


def test_watchdog_and_edge_cases():
    from paper_2606_10440_b200 import Engine, AstraError
    topo, coll, gpu = configs.config1().point(0)
    w = _single(topo, coll, gpu, max_cycles=1000)
    gpu_res, ora = check_workload(w)
    assert gpu_res[0][0].status == 1
    with Engine() as eng:
        eng.run_batch([], 100)                                   # empty batch
        with pytest.raises(AstraError) as ei:
            eng.read_results(0)
        assert ei.value.code == -6
        t = eng.load_infragraph(topo.n_gpus, 0, topo.node_latency, topo.row_ptr, topo.head, topo.bw_q8, topo.latency)
        c = eng.load_collective(coll.n_gpus, coll.owner, coll.dst, coll.lines, coll.cu_lo, coll.cu_n,
                                coll.dep_ptr, coll.dep_step, coll.dep_kind)
        g_small = eng.set_gpu(2, 2, 16, 8)                       # CU range [0,4) exceeds 2 CUs
        with pytest.raises(AstraError) as ei:
            eng.run_batch([(t, c, g_small)], 1000)
        assert ei.value.code == -1
        line3 = T.Topology.from_edges(3, 0, [0, 0, 0], [(0, 1, 256, 5), (1, 0, 256, 5)])
        t3 = eng.load_infragraph(3, 0, line3.node_latency, line3.row_ptr, line3.head, line3.bw_q8, line3.latency)
        c3 = C.single_transfer(3, 0, 2, 4, 0, 1)
        c3id = eng.load_collective(3, c3.owner, c3.dst, c3.lines, c3.cu_lo, c3.cu_n, c3.dep_ptr, c3.dep_step, c3.dep_kind)
        g1 = eng.set_gpu(1, 1, 4, 1)
        with pytest.raises(AstraError) as ei:
            eng.run_batch([(t3, c3id, g1)], 1000)
        assert ei.value.code == -4                               # unreachable
