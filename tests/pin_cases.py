"""Builds the small hand-traced cases of tests/golden/pins_survey_8c.json (round-2 entries G1-G3)
as engine/oracle inputs.  Input construction only: no expected value is computed here."""
import json
import os

from astra_inputs import GpuCfg, collectives as C, topologies as T
from astra_inputs.types import CollectiveBuilder

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "pins_survey_8c.json")))
ROUND2 = ["G1_grant_order_H2", "G1_grant_order_H1", "G1_grant_order_K1", "G2_credit_096", "G2_credit_384",
          "G3_dep_issued", "G3_dep_acked"]
PER_CU = ["H1_issue_per_cu", "H2_cap_per_cu", "H3_issue_and_cap_per_cu"]


def build(key):
    s = GOLD[key]["setup"]
    topo = T.line(2, s["bw_q8"], s["latency"])
    if "steps" in s:
        b = CollectiveBuilder(2, key)
        for owner, dst, lines, cu_lo, cu_n, deps in s["steps"]:
            b.add(owner, dst, lines, cu_lo, cu_n, [tuple(d) for d in deps])
        coll = b.build()
    else:
        coll = C.single_transfer(2, 0, 1, s["lines"], 0, s["cus"])
    return topo, coll, GpuCfg(s["cus"], s["wpc"], s["k"], s["h"], s.get("mode", 0))
