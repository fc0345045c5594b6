"""The no-allocation entry point (include/astra.h: astra_pack_point + astra_run_packed_noalloc): one design point
on one CTA with the engine's scratch in the library's static device array.  Its outputs must equal, bit for bit
(every output is an integer: the tolerance of all parity tests here is 0), those of the existing path
(astra_run_batch + astra_read_results) -- on calls in a row that reuse the array with another point's leftovers in it.
Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

from astra_inputs import configs

pytestmark = pytest.mark.gpu


def _existing_path(eng, point, max_cycles):
    eng.run_batch([point], max_cycles)
    return eng.read_results(0)


def _assert_same(got, ref, label):
    (gs, gts, gll), (rs, rts, rll) = got, ref
    assert (gs.status, gs.n_steps, gs.n_links, gs.window, gs.completion_cycle, gs.total_lines) == \
           (rs.status, rs.n_steps, rs.n_links, rs.window, rs.completion_cycle, rs.total_lines), label
    assert (gts == rts).all(), f"{label}: step timestamps differ"
    assert (gll == rll).all(), f"{label}: link counts differ"


def test_no_alloc_entry_point_matches_existing_path():
    import torch
    from paper_2606_10440_b200 import Engine
    from paper_2606_10440_b200.binding import AstraError, NOALLOC_SCRATCH_BYTES

    dev = torch.device("cuda", 0)
    w1 = configs.config1()                                                   # 4 GPUs, ring all-reduce, 49,152 lines
    w2 = configs.random_workload(7, n_points=3, max_gpus=6, max_steps=24, max_lines=200)
    w3 = configs.config2(range(6, 7))                                        # 8 GPUs on a switch, 9 nodes on one CTA
    with Engine(0) as eng:
        cases = []
        for w in (w1, w2, w3):
            pts = eng.load_workload(w)
            for i, p in enumerate(pts):
                cases.append((f"{w.name}[{i}]", p, w.max_cycles))
        ref = [_existing_path(eng, p, mc) for _, p, mc in cases]
        assert ref[0][0].status == 0 and ref[0][0].completion_cycle == 38623    # config 1 (pin P4)

        # set-up: pack every point, copy the inputs to device memory of ours, allocate the outputs
        packed = []
        for label, p, mc in cases:
            info, buf = eng.pack_point(p, mc)
            assert info.scratch_bytes <= NOALLOC_SCRATCH_BYTES, label
            d_in = torch.from_numpy(buf).to(dev)
            d_out = torch.full((info.out_bytes,), 0xAB, dtype=torch.uint8, device=dev)
            assert d_in.data_ptr() % 256 == 0 and d_out.data_ptr() % 256 == 0
            packed.append((info, d_in, d_out))
        stream = torch.cuda.current_stream().cuda_stream

        def run(j):
            info, d_in, d_out = packed[j]
            d_out.fill_(0xAB)
            eng.run_packed_noalloc(info, d_in.data_ptr(), d_out.data_ptr(), stream)
            torch.cuda.synchronize()
            return Engine.unpack_results(info, d_out.cpu().numpy())

        run(0)                                                               # warm-up (module / kernel already loaded by pack)
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        # calls in a row on the same array: the same point twice, then every other point, then the first again
        order = [0, 0] + list(range(1, len(cases))) + [0]
        for j in order:
            _assert_same(run(j), ref[j], f"no-alloc {cases[j][0]}")
        free1, _ = torch.cuda.mem_get_info()
        assert free1 >= free0, "device memory was allocated by the no-allocation entry point"

        # two calls queued back to back on one stream without a host sync in between (serialised by the stream)
        for j in (0, 1):
            info, d_in, d_out = packed[j]
            d_out.fill_(0xAB)
            eng.run_packed_noalloc(info, d_in.data_ptr(), d_out.data_ptr(), stream)
        torch.cuda.synchronize()
        for j in (0, 1):
            info, _, d_out = packed[j]
            _assert_same(Engine.unpack_results(info, d_out.cpu().numpy()), ref[j], f"queued {cases[j][0]}")

        # the existing path is untouched by all that
        _assert_same(_existing_path(eng, cases[0][1], cases[0][2]), ref[0], "existing path afterwards")

        # a point whose scratch exceeds the static array is refused with a clear error, nothing is launched
        w4 = configs.config4(256)
        big = max(range(256), key=lambda i: w4.meta[i]["cus"] * w4.meta[i]["wpc"] * w4.meta[i]["k"])
        pts4 = eng.load_workload(configs.config4(1, indices=[big]))
        info4, buf4 = eng.pack_point(pts4[0], w4.max_cycles)
        assert info4.scratch_bytes > NOALLOC_SCRATCH_BYTES
        d_in4 = torch.from_numpy(buf4).to(dev)
        d_out4 = torch.zeros(info4.out_bytes, dtype=torch.uint8, device=dev)
        with pytest.raises(AstraError) as ei:
            eng.run_packed_noalloc(info4, d_in4.data_ptr(), d_out4.data_ptr(), stream)
        assert ei.value.code == -5 and "exceeds" in str(ei.value)
        info4.magic = 0
        with pytest.raises(AstraError) as ei:
            eng.run_packed_noalloc(info4, d_in4.data_ptr(), d_out4.data_ptr(), stream)
        assert ei.value.code == -1
