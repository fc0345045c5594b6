#!/usr/bin/env python
"""bench.py -- simulated 128 B cache-line transactions/sec and design points/sec of the CUDA engine on
BASELINE config 4: the 4,096-point design-space sweep (16-GPU ring / 4x4 torus, ring / direct / double
binary tree / halving-doubling all-reduce, 4 KiB .. 16 MiB), one batch, one kernel launch per step.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

One "step" = one pass of the whole hot path (A0 excluded, A1-A8 included: state init, every simulated
lookahead window, result write-out) over the batch.  `value` is measured with the tables resident in
HBM (CUDA events on the launching stream, 256 MiB L2 flush between iterations); `e2e` goes through the
C-ABI from HOST arrays: load_infragraph + load_collective + set_gpu + run_batch + read_results, with
the host<->device copies inside the timed region.

N > 1 (torchrun, one rank per GPU): the job is the first 4,096 x N points of the same seeded sweep,
partitioned by paper_2606_10440_b200.shard (longest-first greedy, no collective on the data path), so
per-GPU work stays fixed ("weak"); time = max over ranks, value = all ranks' transactions / that time.

`other_workloads` carries configs 2, 3 and 5 at full size (>= 3 timed repeats each, same flush), with
their own algorithmic bytes and roofline fraction.  `--impl reference` times the CPU oracle (oracle/)
as it stands on the host cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "simulated_128B_cacheline_transactions_per_sec"
UNIT = "transactions/s"
BYTES_PER_TX_BASE, BYTES_PER_HOP = 72, 20          # SURVEY.md 8(d) algorithmic bytes per transaction
POINTS_PER_GPU = 4096


def get_workload(name: str, n_points: int = POINTS_PER_GPU, indices=None):
    from astra_inputs import configs
    if name == "config4":
        return configs.config4(n_points, indices=indices)
    return configs.by_name(name)


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def engine_source_sha256() -> str:
    """Digest of the engine's sources: profiles/traffic.json is valid for exactly one such digest."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2606_10440_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cpp", ".h", ".cuh")):
            h.update(f.encode()); h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()


def profiled_traffic(workload_name: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one astra_step_kernel launch from the committed
    `ncu --set full` summary (profiles/traffic.json), or None when that capture was taken on other
    engine sources than the ones running now."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        t = json.load(open(p))
        if t.get("engine_source_sha256") == engine_source_sha256():
            return t.get("dram_bytes_per_launch", {}).get(workload_name)
    except Exception:
        pass
    return None


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


class ClockSampler(threading.Thread):
    """Samples nvidia-smi SM clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def run(self):
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self._stop_evt.wait(0.2)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=6)
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        mx = [int(r[1]) for r in self.rows if len(r) > 1 and r[1].isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows for i in range(4) if len(r) > 2 + i and r[2 + i].startswith("Active")})
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


# ---------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline, --impl reference): the only places that execute oracle/
# ---------------------------------------------------------------------------------------------
def oracle_sample(w, stride: int, offset: int = 0):
    """A bounded, size-stratified sample of a workload's design points: every `stride`-th point in
    index order from `offset` (the sweep is seeded uniformly, so a stride keeps the size / parameter mix)."""
    return list(range(min(offset, max(0, w.n_points - 1)), w.n_points, max(1, stride)))


def oracle_time(w, sample, cores: int):
    from oracle import oracle
    oracle.build()
    t0 = time.perf_counter()
    res = oracle.run_workload(w, sample, processes=cores)          # plain scan, one point per process
    dt = time.perf_counter() - t0
    lines = sum(r.total_lines for r in res)
    return lines, dt


# The oracle's plain scan visits every wavefront of every GPU in every cycle: on the config-4 sweep (up to 4,096
# wavefronts per GPU, up to 9 M cycles per point) a design point costs it between a fraction of a second and ~8
# minutes of one core, ~23 core-hours for the 4,096 points.  The bounded sample is every 256th point from point 3
# (16 points, 10.8 M transactions, longest point ~35 s); the one-core figure uses its first four points.
C4_STRIDE, C4_OFFSET, C4_ONE_CORE_POINTS = 256, 3, 4


def oracle_baseline(w):
    """The oracle as it stands (plain scan) on the box's host cores: all cores with one design point per
    process, and one core, each on a bounded sample of the same workload."""
    cores = max(1, min(os.cpu_count() or 1, 64))
    if w.n_points >= 1024:
        sa = oracle_sample(w, C4_STRIDE, C4_OFFSET)
        s1 = sa[:C4_ONE_CORE_POINTS]
        what = f"every {C4_STRIDE}th design point of {w.name} from point {C4_OFFSET}"
    else:
        sa = oracle_sample(w, 1)
        s1 = sorted(sa, key=lambda i: w.collectives[w.points[i][1]].total_lines)[:max(1, len(sa) // 2)]
        what = f"all design points of {w.name}"
    lines_a, dt_a = oracle_time(w, sa, min(cores, len(sa)))
    lines_1, dt_1 = oracle_time(w, s1, 1)
    return {"value": lines_a / dt_a, "unit": UNIT, "cores": min(cores, len(sa)), "kind": "oracle",
            "sample": f"{what}: {len(sa)} of {w.n_points} points, {lines_a} transactions, plain scan, one point per "
                      f"process, {dt_a:.2f} s wall",
            "design_points_per_sec": len(sa) / dt_a,
            "one_core": {"value": lines_1 / dt_1, "unit": UNIT, "design_points_per_sec": len(s1) / dt_1,
                         "sample": f"{len(s1)} points of that sample ({s1}), {lines_1} transactions, {dt_1:.2f} s"},
            "cpu_model": cpu_model(), "host_cores": os.cpu_count(), "seconds": dt_a}


def run_reference(args):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    w = get_workload(args.workload)
    # each step a bounded sample: config 4 -> the cpu_baseline sample without its longest point's class (every 512th
    # point from 3: 8 points), other configs -> all points
    sample = oracle_sample(w, 2 * C4_STRIDE, C4_OFFSET) if w.n_points >= 1024 else oracle_sample(w, 1)
    cores = max(1, min(os.cpu_count() or 1, len(sample), 64))
    for _ in range(1 if args.warmup else 0):
        oracle_time(w, sample[:1], 1)
    runs = [oracle_time(w, sample, cores) for _ in range(max(1, args.steps))]
    lines = runs[0][0]
    dt = sum(r[1] for r in runs) / len(runs)
    val = lines / dt
    desc = (f"{len(sample)} of {w.n_points} design points of {w.name} per step ({sample if len(sample) <= 16 else 'all'}), "
            f"{lines} transactions, plain scan, one point per process")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": w.name, "design_points": w.n_points, "sample": desc},
        "design_points_per_sec": len(sample) / dt,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                         "cpu_model": cpu_model(), "host_cores": os.cpu_count()},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ---------------------------------------------------------------------------------------------
# engine legs
# ---------------------------------------------------------------------------------------------
def algorithmic_bytes(eng, n_points: int, total_lines: int) -> int:
    hops = 0
    for i in range(n_points):
        hops += int(eng.read_results(i, False, True)[2].sum())
    return BYTES_PER_TX_BASE * total_lines + BYTES_PER_HOP * hops


def check_closed_forms(w, summaries):
    """Bench-path spot check against closed forms that hold for the workload (no oracle call here):
    config 2 ring points 14(350 + ceil(n/4)) + 350."""
    if w.name != "config2":
        return
    for s, m in zip(summaries, w.meta):
        if m["algo"] == "ring":
            n = m["lines"] // 8
            assert s.completion_cycle == 14 * (350 + -(-n // 4)) + 350, "config 2 ring closed form violated"


def time_workload(eng, pts, w, stream, flush, steps: int):
    """`steps` timed launches with an L2 flush before each; device time per launch from the engine's own
    CUDA events on its stream."""
    ms = []
    for _ in range(steps):
        flush.zero_()
        eng.run_batch(pts, w.max_cycles, asynchronous=True)
        eng.sync()
        ms.append(eng.last_run_info()[0])
    return ms


def extra_workloads(device, stream, flush, peak):
    """Configs 2, 3, 5 at full size: one preparing run, one warm-up, three timed repeats with the L2
    flush; device time of the engine's launch, algorithmic bytes from the run's own link counts."""
    import numpy as np
    from astra_inputs import configs
    from paper_2606_10440_b200 import Engine
    out = {}
    for name, make in (("config2", configs.config2), ("config3", configs.config3), ("config5", configs.config5)):
        w = make()
        with Engine(device) as eng:
            eng.set_stream(stream.cuda_stream)
            pts = eng.load_workload(w)
            eng.run_batch(pts, w.max_cycles)
            summ = [eng.read_results(i, False, False)[0] for i in range(len(pts))]
            ok = all(s.status == 0 for s in summ)
            check_closed_forms(w, summ)
            alg = algorithmic_bytes(eng, len(pts), w.total_lines())
            time_workload(eng, pts, w, stream, flush, 1)
            ms = time_workload(eng, pts, w, stream, flush, 3)
        k_ms = float(np.mean(ms))
        ach = alg / (k_ms * 1e-3) / 1e9
        out[name] = {"design_points": w.n_points, "transactions": w.total_lines(), "kernel_ms": k_ms, "kernel_ms_runs": ms,
                     "transactions_per_sec": w.total_lines() / (k_ms * 1e-3),
                     "design_points_per_sec": w.n_points / (k_ms * 1e-3), "all_points_finished": ok,
                     "algorithmic_bytes_per_launch": alg,
                     "roofline": {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                                  "traffic": profiled_traffic(name)}}
    return out


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the engine has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    from paper_2606_10440_b200 import Engine, build as engine_build, shard
    engine_build.build()

    # ---- this rank's share of the job (N = 1: the whole config) ----
    if world > 1 and args.workload == "config4":
        from astra_inputs import configs
        n_job = POINTS_PER_GPU * world
        costs = [float(configs.config4_params(i)["lines"]) for i in range(n_job)]
        mine = shard.shard_points(costs, world)[rank]
        w = get_workload("config4", indices=mine)

        class job:                       # what run_sharded needs to know about the whole job
            n_points = n_job
    else:
        n_job = None
        w = get_workload(args.workload)          # single-point configs: replicas only
    total_lines = w.total_lines()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def allsum(x):
        if world == 1:
            return x
        t = torch.tensor([float(x)], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    def allmax(x):
        if world == 1:
            return x
        t = torch.tensor([float(x)], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    stream = torch.cuda.Stream()            # a real (non-default) stream shared by torch and the engine
    torch.cuda.set_stream(stream)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    eng = Engine(local_rank)
    eng.set_stream(stream.cuda_stream)
    pts = eng.load_workload(w)
    eng.run_batch(pts, w.max_cycles)                                     # prepares the batch (A0) + 1 run
    summ = [eng.read_results(i, False, False)[0] for i in range(len(pts))]
    assert all(s.status == 0 for s in summ), "a design point did not finish"
    check_closed_forms(w, summ)
    alg_bytes = algorithmic_bytes(eng, len(pts), total_lines)
    busy = sum(s.busy_cycles for s in summ)

    for _ in range(max(0, args.warmup - 1)):
        flush.zero_()
        eng.run_batch(pts, w.max_cycles)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record(stream)
    kernel_ms = time_workload(eng, pts, w, stream, flush, args.steps)    # L2 flush before every launch
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms_per_step = allmax(ev0.elapsed_time(ev1)) / args.steps
    job_lines = allsum(total_lines)
    job_points = allsum(w.n_points)
    value = job_lines / (ms_per_step * 1e-3)
    k_ms = float(np.mean(kernel_ms))
    _, launches, dev_bytes = eng.last_run_info()
    eng.close()

    # ---- end to end through the C-ABI from host arrays (sharded at N > 1) ----
    def simulate(wl, indices):
        with Engine(local_rank) as e2:
            p2 = e2.load_workload(wl)
            e2.run_batch([p2[i] for i in indices], wl.max_cycles)
            res = [e2.read_results(i) for i in range(len(indices))]
            simulate.bytes = e2.last_transfer_bytes()
        return [(r[0].status, r[0].completion_cycle) for r in res]

    e2e_times = []
    for _ in range(min(3, max(1, args.steps))):
        barrier()
        t0 = time.perf_counter()
        if n_job:       # the N > 1 path: shard.run_sharded partitions, runs this rank's share, gathers every point's result
            outs = shard.run_sharded(job, lambda _job, idx: simulate(w, range(len(idx))), rank, world, costs=costs)
        else:
            outs = simulate(w, range(w.n_points))
        torch.cuda.synchronize()
        e2e_times.append(time.perf_counter() - t0)
        assert all(o[0] == 0 for o in outs)
    e2e_s = allmax(min(e2e_times))
    h2d, d2h = simulate.bytes

    peak, peak_src = measured_peak_gbs()
    achieved = alg_bytes / (k_ms * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic",
        "config": {"workload": w.name, "design_points": int(job_points), "transactions_per_step": int(job_lines),
                   "l2": "256 MiB device write between timed iterations (inside the timed region)",
                   "parallelism": (f"design points sharded over {world} GPU(s) by shard.shard_points, no collective"
                                   if n_job else f"{world} replica(s)")},
        "design_points_per_sec": job_points / (ms_per_step * 1e-3),
        "gpu_launches": launches * args.steps,
        "clocks": clocks,
        "e2e": {"value": job_lines / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "seconds_per_step": e2e_s,
                "design_points_per_sec": job_points / e2e_s},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": profiled_traffic(w.name), "kernel": "astra_step_kernel", "kernel_ms": k_ms,
                     "algorithmic_bytes_per_launch": alg_bytes, "peak_source": peak_src,
                     "note": "bytes = 72 per transaction + 20 per link hop (SURVEY 8(d)), rank 0's launch; the live state "
                             "of a design point sits in shared memory / L2, the kernel is bound by the dependent chain per "
                             "lookahead window, see DESIGN.md section 6; traffic is null unless profiles/traffic.json was "
                             "captured on these engine sources",
                     "node_cycles_stepped": busy, "device_bytes": dev_bytes},
    }
    if rank == 0 and world == 1 and not args.no_extras:
        line["other_workloads"] = extra_workloads(local_rank, stream, flush, peak)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = {k: v for k, v in oracle_baseline(w).items() if k != "seconds"}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the timed runs of configs 2, 3, 5")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
