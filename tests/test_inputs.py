"""Structural checks of the seeded input generators (astra_inputs): they hold no method
arithmetic, so these only check shapes, validity of the DAGs and determinism of the seeds."""
import numpy as np

from astra_inputs import collectives as C, configs
from astra_inputs.types import DEP_DELIVERED


def _check_collective(c, cus):
    S = c.n_steps
    assert c.dep_ptr[0] == 0 and c.dep_ptr[-1] == len(c.dep_step)
    for s in range(S):
        assert c.owner[s] != c.dst[s] and c.lines[s] >= 1 and c.cu_n[s] >= 1
        assert c.cu_lo[s] + c.cu_n[s] <= cus
        for i in range(int(c.dep_ptr[s]), int(c.dep_ptr[s + 1])):
            p, k = int(c.dep_step[i]), int(c.dep_kind[i])
            assert p < s
            if k == DEP_DELIVERED:
                assert c.dst[p] == c.owner[s]
            else:
                assert c.owner[p] == c.owner[s]


def test_config_sizes_match_survey_table():
    assert configs.config1().total_lines() == 49152
    w2 = configs.config2()
    assert w2.n_points == 22 and w2.total_lines() == 29345792
    assert all(c.n_steps == 112 for c in w2.collectives)
    w3 = configs.config3()
    assert w3.collectives[0].n_steps == 1792 and w3.total_lines() == 264241152
    assert (w3.topologies[0].n_nodes, w3.topologies[0].n_links) == (84, 320)
    w5 = configs.config5()
    assert w5.collectives[0].n_steps == 65280
    assert (w5.topologies[0].n_nodes, w5.topologies[0].n_links) == (296, 1024)
    assert int(w5.collectives[0].lines.max()) <= 32768 and int(w5.collectives[0].lines.min()) >= 1


def test_all_configs_valid_dags():
    for w in (configs.config1(), configs.config2(range(6, 8)), configs.config3(8 * 1024),
              configs.config4(64), configs.config5(n_nodes=2)):
        for i in range(w.n_points):
            _, c, g = w.point(i)
            _check_collective(c, g.cus)


def test_config4_seeded_and_in_range():
    a, b = configs.config4(32), configs.config4(32)
    for x, y in zip(a.collectives, b.collectives):
        assert (x.lines == y.lines).all() and (x.dst == y.dst).all()
    for m in a.meta:
        assert m["bw_q8"] in (64, 128, 256, 512, 1024, 2048) and 50 <= m["latency"] <= 2000
        assert 8 <= m["cus"] <= 256 and 1 <= m["wpc"] <= 16 and 4 <= m["k"] <= 64
        assert 32 <= m["lines"] <= 131072


def test_allreduce_volume_per_algorithm():
    n, m = 16, 1000
    assert C.ring_allreduce(n, m, 8)[0].total_lines == 2 * (n - 1) * m
    assert C.direct_allreduce(n, m, 16).total_lines == 2 * (n - 1) * m
    hd = C.halving_doubling_allreduce(n, m, 8)
    # reduce-scatter moves m*(n-1)/n per GPU in total (up to rounding), all-gather the same
    assert abs(hd.total_lines - 2 * (n - 1) * m) <= 2 * n * 4
    dbt = C.double_binary_tree_allreduce(n, m, 8)
    assert dbt.total_lines == 2 * (n - 1) * m     # each tree: (n-1) edges x lines_t, up and down


def test_dbt_each_rank_is_leaf_in_exactly_one_tree():
    for n in (4, 8, 16, 32):
        par = C.dbt_parents(n)
        for t in range(2):
            assert sum(1 for p in par[t] if p < 0) == 1
            children = [[] for _ in range(n)]
            for r, p in enumerate(par[t]):
                if p >= 0:
                    children[p].append(r)
            assert all(len(c) <= 2 for c in children)
        leaf = [[all(p != r for p in par[t]) for r in range(n)] for t in range(2)]
        assert all(leaf[0][r] != leaf[1][r] for r in range(n))


def test_full_size_golden_file_is_complete():
    """tests/golden/full_size.json (written by tests/golden/make_full_size.py from the oracle) holds a digest
    record for config 3, config 5 and every one of the 4,096 config-4 points, and a sample of them is
    reproduced by the oracle here (cheapest points, both scans)."""
    import hashlib
    import json
    import os
    import numpy as np
    from oracle import oracle
    path = os.path.join(os.path.dirname(__file__), "golden", "full_size.json")
    gold = json.load(open(path))
    assert set(gold["config3"]) == {"0"} and set(gold["config5"]) == {"0"}
    assert set(gold["config4"]) == {str(i) for i in range(4096)}
    for rec in list(gold["config4"].values()) + [gold["config3"]["0"], gold["config5"]["0"]]:
        status, completion, total, h_ts, h_ll, scan = rec
        assert status == 0 and completion > 0 and total > 0 and len(h_ts) == 64 and len(h_ll) == 64 and scan in ("plain", "pruned")
    assert gold["config3"]["0"][2] == 264241152 and gold["config3"]["0"][5] == "plain" and gold["config5"]["0"][5] == "plain"
    cheap = sorted(range(4096), key=lambda i: gold["config4"][str(i)][2])[:12]
    for i in cheap:
        topo, coll, gpu, _ = configs.config4_point(i)
        for flags in (0, oracle.FLAG_PRUNED_SCAN):
            r = oracle.run_point(topo, coll, gpu, max_cycles=1 << 26, flags=flags)
            dig = lambda a: hashlib.sha256(np.ascontiguousarray(a, dtype="<u8").tobytes()).hexdigest()
            assert [r.status, r.completion, r.total_lines, dig(r.step_ts), dig(r.link_lines)] == gold["config4"][str(i)][:5]
