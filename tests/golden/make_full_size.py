"""Writes tests/golden/full_size.json: the CPU oracle's results for BASELINE configs 3, 4 (all 4,096
design points) and 5 at FULL size, as per-point digests the -m gpu tests compare the CUDA engine with.

TEST INFRASTRUCTURE.  Imports only `oracle/` and `astra_inputs/` (the seeded generators); nothing
from the CUDA package.  No value in the file comes from the CUDA path.  Run from the repo root:

    python tests/golden/make_full_size.py [--configs 3 4 5] [--processes 8] [--plain-visits 3e9]

Per design point the file holds
    [status, completion_cycle, total_lines, sha256(step_ts), sha256(link_lines), scan]
where step_ts is the oracle's [S,4] u64 array (release, issued, delivered, acked; TS_NONE where
never stamped) and link_lines its [E] u64 array, both hashed as little-endian C-contiguous bytes.

`scan` says which phase-D scan of the oracle produced the digests (oracle/astra_oracle.c header):
  "plain"  the default scan over every wavefront; where it was run, the pruned scan was run too and
           the two results were compared element by element before anything was written;
  "pruned" ORACLE_FLAG_PRUNED_SCAN only: the plain scan's cost (cycles x wavefronts) was above
           --plain-visits for this point.  The pruned scan visits a subset of wavefronts and runs
           the same full check on each; tests/test_oracle_invariants.py proves it equal to the plain
           scan on small cases and this script does so on every point marked "plain".
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import sys
import time

import numpy as np

_ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, _ROOT)

from astra_inputs import configs  # noqa: E402
from oracle import oracle  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "full_size.json")


def digest(arr: np.ndarray) -> str:
    a = np.ascontiguousarray(arr, dtype="<u8")
    return hashlib.sha256(a.tobytes()).hexdigest()


def _one(args):
    cfg, i, plain_visits = args
    if cfg == 4:
        topo, coll, gpu, _ = configs.config4_point(i)
        max_cycles = 1 << 26
    else:
        w = configs.config3() if cfg == 3 else configs.config5()
        topo, coll, gpu = w.point(0)
        max_cycles = w.max_cycles
    t0 = time.time()
    pr = oracle.run_point(topo, coll, gpu, max_cycles=max_cycles, flags=oracle.FLAG_PRUNED_SCAN)
    cycles = int(pr.stats[0])
    cost = cycles * topo.n_gpus * gpu.cus * gpu.wavefronts_per_cu
    scan = "pruned"
    if cost <= plain_visits:
        pl = oracle.run_point(topo, coll, gpu, max_cycles=max_cycles, flags=0)
        assert pl.status == pr.status and pl.completion == pr.completion
        assert (pl.step_ts == pr.step_ts).all() and (pl.link_lines == pr.link_lines).all()
        pr, scan = pl, "plain"
    rec = [int(pr.status), int(pr.completion), int(pr.total_lines), digest(pr.step_ts),
           digest(pr.link_lines), scan]
    return cfg, i, rec, time.time() - t0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="+", default=[3, 4, 5])
    ap.add_argument("--processes", type=int, default=os.cpu_count() or 1)
    ap.add_argument("--plain-visits", type=float, default=3e9,
                    help="run the plain scan too where cycles x wavefronts is at most this")
    ap.add_argument("--points", type=int, default=4096, help="config 4: first N points")
    a = ap.parse_args()

    data = {}
    if os.path.exists(OUT):
        with open(OUT) as f:
            data = json.load(f)
    data["_about"] = ("oracle digests at full size; written by tests/golden/make_full_size.py "
                      "(oracle + astra_inputs only); see that file for the format")

    tasks = []
    for cfg in a.configs:
        if cfg == 4:
            # dearest first so that the pool drains evenly
            pts = sorted(range(a.points), key=lambda i: -configs.config4_point(i)[1].total_lines)
            tasks += [(4, i, a.plain_visits) for i in pts]
        else:
            # one huge point: the plain scan is affordable (minutes), always take it
            tasks.append((cfg, 0, float("inf")))
    oracle.build()
    import multiprocessing as mp
    t0 = time.time()
    done = 0
    with mp.get_context("fork").Pool(a.processes) as pool:
        for cfg, i, rec, dt in pool.imap_unordered(_one, tasks, chunksize=1):
            key = f"config{cfg}"
            data.setdefault(key, {})[str(i)] = rec
            done += 1
            if done % 256 == 0 or cfg != 4:
                print(f"[{time.time() - t0:7.0f}s] {done}/{len(tasks)} config{cfg}[{i}] {rec[5]} {dt:.1f}s",
                      flush=True)
    for key in ("config3", "config4", "config5"):
        if key in data:
            data[key] = {k: data[key][k] for k in sorted(data[key], key=int)}
    tmp = OUT + ".tmp"
    with open(tmp, "w") as f:
        f.write("{\n")
        keys = list(data)
        for n, key in enumerate(keys):
            if isinstance(data[key], dict):
                f.write(f' "{key}": {{\n')
                items = list(data[key].items())
                for m, (k, v) in enumerate(items):
                    f.write(f'  "{k}": {json.dumps(v)}{"," if m + 1 < len(items) else ""}\n')
                f.write(" }")
            else:
                f.write(f' "{key}": {json.dumps(data[key])}')
            f.write(",\n" if n + 1 < len(keys) else "\n")
        f.write("}\n")
    os.replace(tmp, OUT)
    print(f"wrote {OUT} in {time.time() - t0:.0f}s")


if __name__ == "__main__":
    main()
