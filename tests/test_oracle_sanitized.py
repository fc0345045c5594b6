"""The oracle under -fsanitize=address,undefined: oracle/astra_oracle.c is
compiled together with a small file-reading driver (tests/oracle_file_driver.c) into a sanitized
executable, run on config 1, on hand-traced pins and on random workloads with all dependency kinds,
and its output compared with the regular build.  Any heap overflow, use after free, leak, signed
overflow or misaligned access in the oracle fails the run."""
import os
import subprocess

import numpy as np
import pytest

from astra_inputs import configs
from oracle import oracle
from tests import pin_cases

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)


@pytest.fixture(scope="module")
def sanitized_exe(tmp_path_factory):
    exe = str(tmp_path_factory.mktemp("asan") / "oracle_asan")
    cmd = ["gcc", "-O1", "-g", "-std=c11", "-Wall", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-fno-omit-frame-pointer", os.path.join(ROOT, "oracle", "astra_oracle.c"),
           os.path.join(HERE, "oracle_file_driver.c"), "-o", exe]
    try:
        subprocess.check_call(cmd)
    except (subprocess.CalledProcessError, FileNotFoundError) as e:   # no libasan on this machine
        pytest.skip(f"cannot build a sanitized oracle here: {e}")
    return exe


def _dump(path, topo, coll, gpu, max_cycles):
    with open(path, "wb") as f:
        np.array([topo.n_gpus, topo.n_switches, coll.n_steps, len(coll.dep_step), gpu.cus, gpu.wavefronts_per_cu,
                  gpu.max_outstanding, gpu.hbm_lines_per_cycle], dtype="<u4").tofile(f)
        np.array([max_cycles], dtype="<u8").tofile(f)
        for a in (topo.node_latency, topo.row_ptr, topo.head, topo.bw_q8, topo.latency, coll.owner, coll.dst,
                  coll.lines, coll.cu_lo, coll.cu_n, coll.dep_ptr, coll.dep_step):
            np.ascontiguousarray(a, dtype="<u4").tofile(f)
        np.ascontiguousarray(coll.dep_kind, dtype=np.uint8).tofile(f)


def _run(exe, path, flags):
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="halt_on_error=1")
    p = subprocess.run([exe, path, str(flags)], capture_output=True, text=True, env=env, timeout=300)
    assert p.returncode == 0, f"sanitized oracle failed:\n{p.stderr[-3000:]}"
    lines = p.stdout.strip("\n").split("\n")
    status, completion, total = (int(x) for x in lines[0].split())
    ts = np.array([int(x) for x in lines[1].split()], dtype=np.uint64) if len(lines) > 1 else np.zeros(0, np.uint64)
    ll = np.array([int(x) for x in lines[2].split()], dtype=np.uint64) if len(lines) > 2 else np.zeros(0, np.uint64)
    return status, completion, total, ts, ll


def _cases():
    yield "config1", configs.config1().point(0), 1 << 22
    for key in pin_cases.ROUND2:
        yield key, pin_cases.build(key), 1 << 22
    for seed in (3, 11):
        w = configs.random_workload(seed, n_points=3, max_gpus=5, max_steps=16, max_lines=80)
        for i in range(w.n_points):
            yield f"random{seed}[{i}]", w.point(i), w.max_cycles
    topo, coll, gpu = configs.config1().point(0)
    yield "config1_watchdog", (topo, coll, gpu), 1000


@pytest.mark.parametrize("flags", [0, oracle.FLAG_PRUNED_SCAN])
def test_oracle_clean_under_asan_ubsan(sanitized_exe, tmp_path, flags):
    for name, (topo, coll, gpu), max_cycles in _cases():
        path = str(tmp_path / "case.bin")
        _dump(path, topo, coll, gpu, max_cycles)
        status, completion, total, ts, ll = _run(sanitized_exe, path, flags)
        ref = oracle.run_point(topo, coll, gpu, max_cycles=max_cycles, flags=flags)
        assert (status, completion, total) == (ref.status, ref.completion, ref.total_lines), name
        assert (ts == ref.step_ts.reshape(-1)).all() and (ll == ref.link_lines).all(), name
    assert status == 1          # the last case is cut by the watchdog
