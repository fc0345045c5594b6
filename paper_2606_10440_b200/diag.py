"""Per-stage SM clocks of the engine (instrumented build, -DASTRA_DIAG), per CTA and per warp set.

    python -m paper_2606_10440_b200.diag config2 [config3 config4 config5 config1 ...] [--top N]

Builds libastra_b200_diag.so if needed, runs each BASELINE config once to warm up and once for the
numbers, and prints for the most expensive design points the clocks per lookahead window of the
busiest CTAs of the point's group: arrivals + ack discovery, release events, wavefront runs, budget
check / commit, placement, multi-feeder merge, link service, and the wait at the end-of-window barrier.
Diagnostics only: nothing printed here is a benchmark result (the instrumentation costs time).
"""
from __future__ import annotations

import os
import sys

import numpy as np

STAGES = ["arrivals+acks", "release", "wavefront runs", "check/commit", "placement", "merge", "link service", "barrier wait"]


def _sets(d):
    return d[16:].reshape(16, 8).astype(np.int64)


def describe(d) -> str:
    w = max(1, int(d[0]))
    s = _sets(d)
    live = [i for i in range(16) if s[i].sum()]
    if not live:
        return f"windows {int(d[0])}: no nodes on this CTA"
    busy = {i: int(s[i][:7].sum()) // w for i in live}
    b = max(live, key=lambda i: busy[i])
    parts = " ".join(f"{STAGES[j]} {int(s[b][j]) // w}" for j in range(8))
    return (f"windows {int(d[0])} init {int(d[5])} budget-bound GPU-windows {int(d[6])} warp sets {len(live)} "
            f"busy clocks/window max {busy[b]} min {min(busy.values())} | busiest set {b}: {parts}")


def run(name: str, top: int):
    from astra_inputs import configs
    from . import binding, build
    from .binding import Engine
    if binding._LIBPATH != build.LIB_DIAG:              # this process uses the instrumented library
        binding._LIBPATH, binding._lib = build.LIB_DIAG, None
    build.build(diag=True)
    w = configs.by_name(name)
    with Engine(0, 0) as e:
        pts = e.load_workload(w)
        e.run_batch(pts, w.max_cycles)
        e.run_batch(pts, w.max_cycles)
        ms = e.last_run_info()[0]
        print(f"== {name}: {len(pts)} design points, {w.total_lines()} transactions, {ms:.2f} ms (instrumented build)")
        cost = []
        agg = np.zeros(8)
        for i in range(len(pts)):
            d = e.read_diag(i, 0)
            agg += _sets(d)[0]
            cost.append((int(_sets(d)[0].sum()) + int(d[5]), i))
        print("   share of the first warp set's clocks over all points: " +
              ", ".join(f"{STAGES[j]} {100 * agg[j] / max(1.0, agg.sum()):.1f}%" for j in range(8)))
        cost.sort(reverse=True)
        for _, i in cost[:top]:
            s = e.read_results(i, False, False)[0]
            grp = e.point_group(i)
            print(f"   point {i}: completion {s.completion_cycle} lines {s.total_lines} window {s.window} cycles, "
                  f"{grp} CTA(s) {w.meta[i] if i < len(w.meta) else ''}")
            ranks = sorted(range(grp), key=lambda r: -int(_sets(e.read_diag(i, r))[:, :7].sum(axis=1).max()))
            show = ranks[:4] + ([ranks[len(ranks) // 2], ranks[-1]] if grp > 6 else [])
            for r in show:
                print(f"      CTA {r}: {describe(e.read_diag(i, r))}")


def main():
    args = [a for a in sys.argv[1:] if not a.startswith("--")]
    top = 3
    if "--top" in sys.argv:
        top = int(sys.argv[sys.argv.index("--top") + 1]); args = [a for a in args if a != str(top)]
    for name in args or ["config2"]:
        run(name, top)


if __name__ == "__main__":
    main()
