"""ut_decode_static (include/ut_compass.h): the decode with its scratch in the library's built-in device array, for
callers that cannot allocate.  Collected last on purpose (the suite runs with pytest -x).  The existing ut_decode
path is the reference here; it is itself checked against the oracle in test_gpu_parity.py."""
import ctypes as C

import numpy as np
import pytest


@pytest.fixture(scope="module")
def gpu(geom):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from gpu_helpers import GpuRunner
    return GpuRunner(geom)


def container_arrays(gpu, hits, n_events):
    """Everything ut_decode writes for `n_events` events, as numpy (bit patterns for the float arrays)."""
    B = gpu.B
    got, off, st = gpu.hits_numpy(hits, n_events)
    n = int(off[-1])
    out = {f: (a if f == "id" else a.view(np.uint32)) for f, a in got.items()}
    out["hit_offsets"], out["status"] = off, st
    stride = B.ut_sector_offsets_stride(gpu.geom)
    out["x_by_sector"] = hits.x_by_sector[:n].cpu().numpy().view(np.uint32)
    out["idx_by_sector"] = hits.idx_by_sector[:n].cpu().numpy().view(np.uint16)
    out["sector_offsets"] = hits.sector_offsets[:n_events * stride].cpu().numpy().view(np.uint16)
    return out


@pytest.mark.gpu
def test_static_decode_matches_ut_decode_on_two_calls_in_a_row(gpu, wl):
    B, torch = gpu.B, gpu.torch
    # two different batches, so the second call finds the first one's look-back words and counters in the array
    cases = [wl(2, 70), wl(4, 23), wl(2, 70)]
    refs, inputs = [], []
    for geom, b, p in cases:
        hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)        # existing path, own workspace
        refs.append((hits, container_arrays(gpu, hits, b.n_events)))
        inputs.append((B.to_device_raw(b.raw), B.to_device_u32(b.bank_offsets)))
    outs = [B.Hits(b.hit_capacity, max(b.n_events, 1), gpu.geom) for _, b, _ in cases]
    torch.cuda.synchronize()
    for (geom, b, p), (raw_d, bo_d), hits in zip(cases, inputs, outs):              # back to back, one stream, no sync
        B.ut_decode_static(raw_d, bo_d, b.n_events, gpu.geom, hits)
    torch.cuda.synchronize()
    for (geom, b, p), (ref_hits, ref), hits in zip(cases, refs, outs):
        got = container_arrays(gpu, hits, b.n_events)
        assert got["status"] == ref["status"] == 0
        assert int(ref["hit_offsets"][-1]) > 1000
        for k, v in ref.items():
            assert np.array_equal(v, got[k]), k                                     # bit-exact, like the parity tests
        assert not bool(hits.workspace.any())             # the container's own workspace was not handed to the kernel
        # and the container is as usable downstream as the other one
        t_ref, t_got = gpu.compass(ref_hits, b, p), gpu.compass(hits, b, p)
        for k in ("hit_idx", "n_hits"):
            assert np.array_equal(t_ref[k], t_got[k]), k
        for k in ("qop", "chi2"):
            assert np.array_equal(t_ref[k].view(np.uint32), t_got[k].view(np.uint32)), k
        assert t_got["status"] == 0


@pytest.mark.gpu
def test_static_decode_empty_batch(gpu, wl):
    B, torch = gpu.B, gpu.torch
    geom, b, p = wl(2, 5)
    hits = B.Hits(16, 1, gpu.geom)
    hits.hit_offsets.fill_(7)
    B.ut_decode_static(B.to_device_raw(b.raw), B.to_device_u32(b.bank_offsets), 0, gpu.geom, hits)
    torch.cuda.synchronize()
    assert int(hits.hit_offsets[0].item()) == 0 and int(hits.status.item()) == 0


def test_static_decode_rejects_batches_above_its_limit():
    """Host-side check, no GPU needed: nothing is launched, the error text names the limit."""
    from paper_2002_11529_b200 import binding as B
    lib = B._lib
    h = B.ut_hits()
    rc = lib.ut_decode_static(None, None, B.UT_DECODE_STATIC_MAX_EVENTS + 1, None, C.byref(h), None, None)
    assert rc == B.UT_ERR_LIMIT
    text = lib.ut_last_error().decode()
    assert "UT_DECODE_STATIC_MAX_EVENTS" in text and str(B.UT_DECODE_STATIC_MAX_EVENTS) in text
    assert lib.ut_decode_static(None, None, 1, None, None, None, None) == B.UT_ERR_NULL
