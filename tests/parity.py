"""Shared helper for the -m gpu parity tests: run a Workload through the CUDA engine (via the
C-ABI binding) and through the CPU oracle, and compare every integer output bit for bit."""
import numpy as np

from oracle import oracle


def compare_point(res_gpu, res_or, label=""):
    summ, ts, ll = res_gpu
    assert summ.status == res_or.status, f"{label}: status {summ.status} != oracle {res_or.status}"
    # completion = max t_ack over the fully acked steps (R14), whatever the status (a run cut by the watchdog included)
    assert summ.completion_cycle == res_or.completion, \
        f"{label}: completion {summ.completion_cycle} != oracle {res_or.completion}"
    assert summ.total_lines == res_or.total_lines
    bad = np.nonzero((ts != res_or.step_ts).any(axis=1))[0]
    assert bad.size == 0, (f"{label}: {bad.size} steps differ, first {bad[:5].tolist()}: "
                           f"gpu {ts[bad[:5]].astype(np.int64).tolist()} oracle {res_or.step_ts[bad[:5]].astype(np.int64).tolist()}")
    badl = np.nonzero(ll != res_or.link_lines)[0]
    assert badl.size == 0, f"{label}: link_lines differ at {badl[:8].tolist()}"


def check_workload(w, indices=None, flags=0, oracle_flags=0, processes=1, engine_flags=None):
    from paper_2606_10440_b200 import simulate_workload
    idx = list(range(w.n_points)) if indices is None else list(indices)
    gpu = simulate_workload(w, flags=flags, indices=idx)
    ora = oracle.run_workload(w, idx, processes=processes, flags=oracle_flags)
    for j, i in enumerate(idx):
        compare_point(gpu[j], ora[j], label=f"{w.name}[{i}] {w.meta[i] if i < len(w.meta) else ''}")
    return gpu, ora
