"""ctypes binding of include/astra.h.  Same call names as the C-ABI; marshalling only -- every
step of the hot path runs in the CUDA kernels of csrc/astra_engine.cu."""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# ASTRA_DIAG=1 in the environment selects the instrumented build (build.build(diag=True)); diagnostics only
_LIBPATH = os.path.join(_HERE, "libastra_b200_diag.so" if os.environ.get("ASTRA_DIAG") == "1" else
                        f"libastra_b200{os.environ.get('ASTRA_LIB_SUFFIX', '')}.so")

EXPORTED_SYMBOLS = [
    "astra_create", "astra_destroy", "astra_last_error", "astra_set_stream",
    "astra_load_infragraph", "astra_load_collective", "astra_set_gpu", "astra_set_gpu_ex",
    "astra_run_batch", "astra_run_batch_async", "astra_sync", "astra_read_results",
    "astra_last_run_info", "astra_last_transfer_bytes", "astra_read_diag", "astra_point_group",
    "astra_pack_point", "astra_run_packed_noalloc",
]
NOALLOC_SCRATCH_BYTES = 16 << 20     # ASTRA_NOALLOC_SCRATCH_BYTES

FLAG_NO_WINDOW_SKIP = 1
FLAG_WINDOW_1 = 2
FLAG_SERIAL_ISSUE = 4          # testing: cycle-serial issue path everywhere
FLAG_SERIAL_ARRIVALS = 8       # testing: one task per in-link
FLAG_NO_HEAVY = 16             # testing: no warp-per-wavefront path
FLAG_NO_PRIORITY_SWEEP = 32    # testing: budget-bound windows on the cycle-serial path
FLAG_RUN_AHEAD = 64            # one-CTA points: nodes run ahead of the nodes they do not depend on (no barrier per window)


def FLAG_WARPS(w: int) -> int:
    """ASTRA_FLAG_WARPS(w): w warps per CTA, 16 / w CTAs per SM."""
    return (w & 0x3F) << 20


def FLAG_GROUP(g: int) -> int:
    """ASTRA_FLAG_GROUP(g): run every design point on a group of g CTAs."""
    return (g & 0xFF) << 8

TS_NONE = np.uint64(0xFFFFFFFFFFFFFFFF)


class AstraError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"astra error {code}: {msg}")
        self.code = code


class _Point(ctypes.Structure):
    _fields_ = [("topo_id", ctypes.c_uint32), ("coll_id", ctypes.c_uint32),
                ("gpu_id", ctypes.c_uint32), ("reserved", ctypes.c_uint32)]


class _Summary(ctypes.Structure):
    _fields_ = [("status", ctypes.c_int32), ("n_steps", ctypes.c_uint32), ("n_links", ctypes.c_uint32),
                ("window", ctypes.c_uint32), ("completion_cycle", ctypes.c_uint64),
                ("total_lines", ctypes.c_uint64), ("busy_cycles", ctypes.c_uint64),
                ("skipped_cycles", ctypes.c_uint64)]


@dataclass
class Summary:
    status: int
    n_steps: int
    n_links: int
    window: int
    completion_cycle: int
    total_lines: int
    busy_cycles: int
    skipped_cycles: int


_lib = None


class PackedInfo(ctypes.Structure):
    """astra_packed_info (include/astra.h)."""
    _fields_ = [("magic", ctypes.c_uint64), ("in_bytes", ctypes.c_uint64), ("out_bytes", ctypes.c_uint64),
                ("scratch_bytes", ctypes.c_uint64), ("off_const", ctypes.c_uint64), ("off_desc", ctypes.c_uint64),
                ("off_order", ctypes.c_uint64), ("off_step_ts", ctypes.c_uint64), ("off_link_lines", ctypes.c_uint64),
                ("off_summary", ctypes.c_uint64), ("n_steps", ctypes.c_uint32), ("n_links", ctypes.c_uint32),
                ("hot_bytes", ctypes.c_uint32), ("warps", ctypes.c_uint32)]


def load_library(path: Optional[str] = None):
    """dlopen the engine.  Raises (loudly) when it has not been built; never falls back."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or _LIBPATH
    if not os.path.exists(p):
        raise FileNotFoundError(f"{p} not built: run `python -m paper_2606_10440_b200.build` "
                                "(or __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(p)
    vp, u32, u64, i32 = ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int32
    lib.astra_create.argtypes = [ctypes.POINTER(vp), i32, u64]
    lib.astra_destroy.argtypes = [vp]
    lib.astra_last_error.argtypes = [vp]
    lib.astra_last_error.restype = ctypes.c_char_p
    lib.astra_set_stream.argtypes = [vp, vp]
    lib.astra_load_infragraph.argtypes = [vp, u32, u32, vp, vp, vp, vp, vp, ctypes.POINTER(u32)]
    lib.astra_load_collective.argtypes = [vp, u32, u32, vp, vp, vp, vp, vp, vp, vp, vp, ctypes.POINTER(u32)]
    lib.astra_set_gpu.argtypes = [vp, u32, u32, u32, u32, ctypes.POINTER(u32)]
    lib.astra_set_gpu_ex.argtypes = [vp, u32, u32, u32, u32, u32, ctypes.POINTER(u32)]
    lib.astra_run_batch.argtypes = [vp, u32, vp, u64]
    lib.astra_run_batch_async.argtypes = [vp, u32, vp, u64]
    lib.astra_sync.argtypes = [vp]
    lib.astra_read_results.argtypes = [vp, u32, ctypes.POINTER(_Summary), vp, vp]
    lib.astra_read_diag.argtypes = [vp, u32, u32, vp]
    lib.astra_point_group.argtypes = [vp, u32, ctypes.POINTER(u32)]
    lib.astra_last_run_info.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(u32), ctypes.POINTER(u64)]
    lib.astra_last_transfer_bytes.argtypes = [vp, ctypes.POINTER(u64), ctypes.POINTER(u64)]
    lib.astra_pack_point.argtypes = [vp, vp, u64, vp, u64, ctypes.POINTER(PackedInfo)]
    lib.astra_run_packed_noalloc.argtypes = [vp, ctypes.POINTER(PackedInfo), vp, vp, vp]
    for name in EXPORTED_SYMBOLS:
        if name != "astra_last_error":
            getattr(lib, name).restype = i32
    if path is None:
        _lib = lib
    return lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _u32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.uint32)


class Engine:
    """One astra_ctx.  Methods mirror the C calls one to one."""

    def __init__(self, device: int = 0, flags: int = 0):
        self._lib = load_library()
        self._ctx = ctypes.c_void_p()
        rc = self._lib.astra_create(ctypes.byref(self._ctx), device, flags)
        if rc:
            self._ctx = None
            raise AstraError(rc, "astra_create failed (no usable CUDA device? there is no CPU fallback)")
        self._points = None
        self._n_points = 0

    def _check(self, rc: int):
        if rc:
            raise AstraError(rc, (self._lib.astra_last_error(self._ctx) or b"").decode())

    def close(self):
        if self._ctx:
            self._lib.astra_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_stream(self, cuda_stream_ptr: int):
        self._check(self._lib.astra_set_stream(self._ctx, ctypes.c_void_p(cuda_stream_ptr)))

    def load_infragraph(self, n_gpus, n_switches, node_latency, row_ptr, head, bw_q8, latency) -> int:
        arrs = [_u32(node_latency), _u32(row_ptr), _u32(head), _u32(bw_q8), _u32(latency)]
        out = ctypes.c_uint32()
        self._check(self._lib.astra_load_infragraph(self._ctx, n_gpus, n_switches, *[_ptr(a) for a in arrs],
                                                    ctypes.byref(out)))
        return out.value

    def load_collective(self, n_gpus, owner, dst, lines, cu_lo, cu_n, dep_ptr, dep_step, dep_kind) -> int:
        arrs = [_u32(owner), _u32(dst), _u32(lines), _u32(cu_lo), _u32(cu_n), _u32(dep_ptr), _u32(dep_step),
                np.ascontiguousarray(dep_kind, dtype=np.uint8)]
        out = ctypes.c_uint32()
        self._check(self._lib.astra_load_collective(self._ctx, n_gpus, len(arrs[0]), *[_ptr(a) for a in arrs],
                                                    ctypes.byref(out)))
        return out.value

    def set_gpu(self, cus, wavefronts_per_cu, max_outstanding, hbm_lines_per_cycle) -> int:
        out = ctypes.c_uint32()
        self._check(self._lib.astra_set_gpu(self._ctx, cus, wavefronts_per_cu, max_outstanding,
                                            hbm_lines_per_cycle, ctypes.byref(out)))
        return out.value

    def set_gpu_ex(self, cus, wavefronts_per_cu, max_outstanding, hbm_lines_per_cycle, mode) -> int:
        out = ctypes.c_uint32()
        self._check(self._lib.astra_set_gpu_ex(self._ctx, cus, wavefronts_per_cu, max_outstanding,
                                               hbm_lines_per_cycle, mode, ctypes.byref(out)))
        return out.value

    def _marshal_points(self, points: Sequence[Tuple[int, int, int]]):
        arr = (_Point * max(1, len(points)))()
        for i, (t, c, g) in enumerate(points):
            arr[i].topo_id, arr[i].coll_id, arr[i].gpu_id, arr[i].reserved = t, c, g, 0
        return arr

    def run_batch(self, points, max_cycles: int, asynchronous: bool = False):
        if not isinstance(points, ctypes.Array):
            self._n_points = len(points)
            points = self._marshal_points(points)
        self._points = points
        fn = self._lib.astra_run_batch_async if asynchronous else self._lib.astra_run_batch
        self._check(fn(self._ctx, self._n_points, ctypes.cast(points, ctypes.c_void_p), max_cycles))

    def sync(self):
        self._check(self._lib.astra_sync(self._ctx))

    def read_results(self, point: int, want_steps: bool = True, want_links: bool = True):
        s = _Summary()
        self._check(self._lib.astra_read_results(self._ctx, point, ctypes.byref(s), None, None))
        step_ts = np.zeros(max(1, 4 * s.n_steps), dtype=np.uint64) if want_steps else None
        link_lines = np.zeros(max(1, s.n_links), dtype=np.uint64) if want_links else None
        if want_steps or want_links:
            self._check(self._lib.astra_read_results(self._ctx, point, ctypes.byref(s), _ptr(step_ts), _ptr(link_lines)))
        summ = Summary(s.status, s.n_steps, s.n_links, s.window, s.completion_cycle, s.total_lines,
                       s.busy_cycles, s.skipped_cycles)
        return (summ,
                step_ts[:4 * s.n_steps].reshape(s.n_steps, 4) if want_steps else None,
                link_lines[:s.n_links] if want_links else None)

    def read_diag(self, point: int, cta_rank: int = 0) -> np.ndarray:
        out = np.zeros(144, dtype=np.uint64)
        self._check(self._lib.astra_read_diag(self._ctx, point, cta_rank, _ptr(out)))
        return out

    def point_group(self, point: int) -> int:
        g = ctypes.c_uint32()
        self._check(self._lib.astra_point_group(self._ctx, point, ctypes.byref(g)))
        return g.value

    def last_run_info(self):
        ms, n, b = ctypes.c_float(), ctypes.c_uint32(), ctypes.c_uint64()
        self._check(self._lib.astra_last_run_info(self._ctx, ctypes.byref(ms), ctypes.byref(n), ctypes.byref(b)))
        return ms.value, n.value, b.value

    def last_transfer_bytes(self):
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        self._check(self._lib.astra_last_transfer_bytes(self._ctx, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    # no-allocation entry point (include/astra.h): set-up, then runs that only clear the scratch header and launch
    def pack_point(self, point: Tuple[int, int, int], max_cycles: int):
        """astra_pack_point: returns (PackedInfo, uint8 host array of info.in_bytes holding the packed inputs)."""
        arr = self._marshal_points([point])
        info = PackedInfo()
        self._check(self._lib.astra_pack_point(self._ctx, ctypes.cast(arr, ctypes.c_void_p), max_cycles, None, 0, ctypes.byref(info)))
        buf = np.zeros(info.in_bytes, dtype=np.uint8)
        self._check(self._lib.astra_pack_point(self._ctx, ctypes.cast(arr, ctypes.c_void_p), max_cycles, _ptr(buf), buf.nbytes, ctypes.byref(info)))
        return info, buf

    def run_packed_noalloc(self, info: PackedInfo, d_in: int, d_out: int, stream: int = 0):
        """astra_run_packed_noalloc: d_in / d_out are device addresses (256-byte aligned), stream a cudaStream_t or 0."""
        self._check(self._lib.astra_run_packed_noalloc(self._ctx, ctypes.byref(info), ctypes.c_void_p(d_in), ctypes.c_void_p(d_out),
                                                       ctypes.c_void_p(stream) if stream else None))

    @staticmethod
    def unpack_results(info: PackedInfo, out: np.ndarray):
        """Host copy of an output buffer -> (Summary, step_ts[S,4], link_lines[E]) as read_results returns them."""
        s = _Summary.from_buffer_copy(out[info.off_summary:info.off_summary + ctypes.sizeof(_Summary)].tobytes())
        ts = out[info.off_step_ts:info.off_step_ts + 32 * info.n_steps].view(np.uint64).reshape(info.n_steps, 4).copy()
        ll = out[info.off_link_lines:info.off_link_lines + 8 * info.n_links].view(np.uint64).copy()
        return (Summary(s.status, s.n_steps, s.n_links, s.window, s.completion_cycle, s.total_lines, s.busy_cycles, s.skipped_cycles),
                ts, ll)

    # convenience over the calls above: load a whole astra_inputs.Workload
    def load_workload(self, w) -> List[Tuple[int, int, int]]:
        tids = [self.load_infragraph(t.n_gpus, t.n_switches, t.node_latency, t.row_ptr, t.head, t.bw_q8, t.latency)
                for t in w.topologies]
        cids = [self.load_collective(c.n_gpus, c.owner, c.dst, c.lines, c.cu_lo, c.cu_n, c.dep_ptr, c.dep_step,
                                     c.dep_kind) for c in w.collectives]
        gids = [self.set_gpu_ex(g.cus, g.wavefronts_per_cu, g.max_outstanding, g.hbm_lines_per_cycle, getattr(g, "mode", 0))
                if getattr(g, "mode", 0) else self.set_gpu(g.cus, g.wavefronts_per_cu, g.max_outstanding, g.hbm_lines_per_cycle)
                for g in w.gpus]
        return [(tids[t], cids[c], gids[g]) for (t, c, g) in w.points]


def simulate_workload(w, device: int = 0, flags: int = 0, indices=None):
    """Load, run and read back a Workload.  Returns [(Summary, step_ts[S,4], link_lines[E])]."""
    with Engine(device, flags) as eng:
        pts = eng.load_workload(w)
        if indices is not None:
            pts = [pts[i] for i in indices]
        eng.run_batch(pts, w.max_cycles)
        return [eng.read_results(i) for i in range(len(pts))]
