"""ctypes wrapper around oracle/astra_oracle.c.

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Never imported by paper_2606_10440_b200.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "astra_oracle.c")
_LIB = os.path.join(_HERE, "libastra_oracle.so")

FLAG_PRUNED_SCAN = 1
FLAG_ISSUE_PER_CU = 2      # R12': one line per CU per cycle
FLAG_CAP_PER_CU = 4        # R2': max_outstanding per CU
TS_NONE = np.uint64(0xFFFFFFFFFFFFFFFF)

TR_ISSUE, TR_ACCEPT, TR_DELIVER, TR_ACK, TR_RELEASE = range(5)

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-Wall", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_run.restype = ctypes.c_int
        _lib.oracle_route.restype = ctypes.c_int
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


@dataclass
class OracleResult:
    status: int
    completion: int
    total_lines: int
    step_ts: np.ndarray      # [S,4] u64: release, issued, delivered, acked
    link_lines: np.ndarray   # [E] u64
    stats: np.ndarray        # [8] u64
    trace: Optional[np.ndarray] = None   # [n,5] u64: cycle, kind, step, gpu*65536+wf, link


def route(topo):
    lib = _load()
    V, G = topo.n_nodes, topo.n_gpus
    dist = np.zeros(V * G, dtype=np.uint64)
    nl = np.zeros(V * G, dtype=np.uint32)
    rc = lib.oracle_route(ctypes.c_uint32(topo.n_gpus), ctypes.c_uint32(topo.n_switches),
                          _p(topo.node_latency), _p(topo.row_ptr), _p(topo.head), _p(topo.bw_q8),
                          _p(topo.latency), _p(dist), _p(nl))
    if rc:
        raise RuntimeError(f"oracle_route failed: {rc}")
    return dist.reshape(V, G), nl.reshape(V, G)


def run_point(topo, coll, gpu, max_cycles: int = 1 << 40, flags: int = 0,
              trace_cap: int = 0, check: bool = True) -> OracleResult:
    lib = _load()
    flags |= 2 * (getattr(gpu, "mode", 0) & 3)          # GpuCfg.mode bit 0: issue per CU, bit 1: cap per CU
    S, E = coll.n_steps, topo.n_links
    step_ts = np.zeros(max(1, 4 * S), dtype=np.uint64)
    link_lines = np.zeros(max(1, E), dtype=np.uint64)
    stats = np.zeros(8, dtype=np.uint64)
    status = ctypes.c_int32(-1)
    completion = ctypes.c_uint64(0)
    total = ctypes.c_uint64(0)
    trace = np.zeros((trace_cap, 5), dtype=np.uint64) if trace_cap else None
    trace_len = ctypes.c_uint64(0)
    rc = lib.oracle_run(
        ctypes.c_uint32(topo.n_gpus), ctypes.c_uint32(topo.n_switches), _p(topo.node_latency),
        _p(topo.row_ptr), _p(topo.head), _p(topo.bw_q8), _p(topo.latency),
        ctypes.c_uint32(S), _p(coll.owner), _p(coll.dst), _p(coll.lines), _p(coll.cu_lo), _p(coll.cu_n),
        _p(coll.dep_ptr), _p(coll.dep_step), _p(coll.dep_kind),
        ctypes.c_uint32(gpu.cus), ctypes.c_uint32(gpu.wavefronts_per_cu),
        ctypes.c_uint32(gpu.max_outstanding), ctypes.c_uint32(gpu.hbm_lines_per_cycle),
        ctypes.c_uint64(max_cycles), ctypes.c_uint32(flags),
        ctypes.byref(status), ctypes.byref(completion), ctypes.byref(total),
        _p(step_ts), _p(link_lines), _p(stats),
        _p(trace), ctypes.c_uint64(trace_cap), ctypes.byref(trace_len))
    if rc and check:
        raise RuntimeError(f"oracle_run failed: {rc}")
    res = OracleResult(status=status.value if rc == 0 else rc, completion=completion.value,
                       total_lines=total.value, step_ts=step_ts[:4 * S].reshape(S, 4),
                       link_lines=link_lines[:E], stats=stats)
    if trace is not None:
        if trace_len.value > trace_cap:
            raise RuntimeError("trace overflow")
        res.trace = trace[:trace_len.value]
    return res


def _run_idx(args):
    w, i, max_cycles, flags = args
    t, c, g = w.point(i)
    return run_point(t, c, g, max_cycles=max_cycles, flags=flags)


def run_workload(w, indices=None, processes: int = 1, flags: int = 0):
    """Run design points of a Workload (single-threaded per point; `processes` points at once)."""
    idx = list(range(w.n_points)) if indices is None else list(indices)
    _load()
    if processes <= 1 or len(idx) <= 1:
        return [_run_idx((w, i, w.max_cycles, flags)) for i in idx]
    import multiprocessing as mp
    with mp.get_context("fork").Pool(processes) as pool:
        return pool.map(_run_idx, [(w, i, w.max_cycles, flags) for i in idx], chunksize=1)
