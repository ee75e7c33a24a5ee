"""-m gpu: a short seeded soak of the CUDA path against the oracle -- contiguous slices of the config-3 and config-4
batches at sizes around the launch thresholds (one CTA per event, split events, more than one wave of CTAs with the
event order, the static decode entry), uneven track counts, random launch tunings.  Every output element bit for bit.
(The same loop ran for 1643 cases / 7 minutes on a B200 at the end of round 2 without a difference.)"""
import dataclasses
import random

import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu(geom):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from gpu_helpers import GpuRunner
    return GpuRunner(geom)


def slice_batch(b, ns, e0, ne):
    bo, vo = b.bank_offsets.astype(np.int64), b.velo_offsets.astype(np.int64)
    r0, r1 = int(bo[e0 * ns]), int(bo[(e0 + ne) * ns])
    v0, v1 = int(vo[e0]), int(vo[e0 + ne])
    return dataclasses.replace(
        b, n_events=ne, raw=b.raw[r0:r1].copy(), bank_offsets=(bo[e0 * ns:(e0 + ne) * ns + 1] - r0).astype(np.uint32),
        velo_x=b.velo_x[v0:v1], velo_y=b.velo_y[v0:v1], velo_tx=b.velo_tx[v0:v1], velo_ty=b.velo_ty[v0:v1],
        velo_offsets=(vo[e0:e0 + ne + 1] - v0).astype(np.uint32), truth_hit_id=b.truth_hit_id[v0:v1],
        truth_q=b.truth_q[v0:v1], truth_p=b.truth_p[v0:v1], n_hits_event=b.n_hits_event[e0:e0 + ne],
        hit_capacity=(r1 - r0 - 6 * ne * ns) // 2)


def thin_tracks(b, rng):
    """Some events lose all or most of their VELO tracks."""
    vo, keep = b.velo_offsets.astype(np.int64), []
    for e in range(b.n_events):
        n = int(vo[e + 1] - vo[e])
        keep.append(np.arange(vo[e], vo[e] + rng.choice((0, n // 5, n, n, n))))
    idx = np.concatenate(keep)
    return dataclasses.replace(
        b, velo_x=b.velo_x[idx], velo_y=b.velo_y[idx], velo_tx=b.velo_tx[idx], velo_ty=b.velo_ty[idx],
        velo_offsets=np.concatenate([[0], np.cumsum([len(k) for k in keep])]).astype(np.uint32),
        truth_hit_id=b.truth_hit_id[idx], truth_q=b.truth_q[idx], truth_p=b.truth_p[idx])


def test_seeded_soak(gpu, wl):
    import torch
    from gpu_helpers import compare_decode, compare_tracks
    B = gpu.B
    rng = random.Random(20260211)
    sizes = {3: (1, 100, 148, 149, 296, 297, 592, 593, 700, 1000), 4: (1, 148, 149, 170, 297)}
    seen_order = seen_static = 0
    try:
        for case in range(36):
            c = 4 if case % 4 == 3 else 3
            geom, full, p = wl(c)
            ne = rng.choice(sizes[c])
            b = slice_batch(full, geom.n_sectors, rng.randrange(0, full.n_events - ne + 1), ne)
            if rng.random() < 0.5:
                b = thin_tracks(b, rng)
            tun = {}
            if rng.random() < 0.4:
                tun["compass_block"] = rng.choice((64, 128, 192, 224, 256, 384, 512, 576, 640))
            if rng.random() < 0.2:
                tun["compass_event_order"] = 0
            if rng.random() < 0.2:
                tun["decode_block"] = rng.choice((128, 256, 384, 512))
            if rng.random() < 0.2:
                tun["compass_split"] = rng.choice((1, 2, 4))
            B.ut_tuning_set(**tun) if tun else B.ut_tuning_set(None)
            h_ref, t_ref = oracle.run_batch(b, geom, p)
            if rng.random() < 0.3:
                hits = B.Hits(b.hit_capacity, max(ne, 1), gpu.geom)
                keep = (B.to_device_raw(b.raw), B.to_device_u32(b.bank_offsets))
                B.ut_decode_static(keep[0], keep[1], ne, gpu.geom, hits)
                torch.cuda.synchronize()
                seen_static += 1
            else:
                hits = gpu.decode(b.raw, b.bank_offsets, ne, b.hit_capacity)
            got, off, st = gpu.hits_numpy(hits, ne)
            compare_decode(h_ref, got, off, st)
            trk = gpu.compass(hits, b, p)
            seen_order += B.last_launch_info()["compass_event_order"] > 0
            n_diff, _ = compare_tracks(t_ref, trk)
            assert n_diff == 0, (case, c, ne, tun)
            assert np.array_equal(trk["chi2"].view(np.uint32), t_ref.chi2.view(np.uint32)), (case, c, ne, tun)
            assert np.array_equal(trk["qop"].view(np.uint32), t_ref.qop.view(np.uint32)), (case, c, ne, tun)
    finally:
        B.ut_tuning_set(None)
    assert seen_order >= 3 and seen_static >= 3          # the paths the soak is there for did run


def test_seeded_pipeline_soak(gpu, wl):
    """ut_pipeline_run_host on slices of the two batches with random chunk sizes and host layouts, twice per pipeline.
    The first case is the one the round-2 soak caught: busy events (config 4) in 3 chunks, where the Compass launches of
    two chunks overlap on different streams -- they must not share a work ticket."""
    import torch
    B = gpu.B
    rng = random.Random(5)
    cases = [(4, 333, {"pipeline_chunk_events": 100}, True)]
    for _ in range(14):
        c = rng.choice((3, 3, 4))
        ne = rng.choice((1, 50, 149, 333, 500, 667, 1000)) if c == 3 else rng.choice((1, 100, 333, 420))
        tun = {"pipeline_chunk_events": rng.choice((40, 100, 250, 333, 500))} if rng.random() < 0.6 else {}
        cases.append((c, ne, tun, rng.random() < 0.6))
    try:
        for c, ne, tun, one in cases:
            geom, full, p = wl(c)
            b = slice_batch(full, geom.n_sectors, rng.randrange(0, full.n_events - ne + 1), ne)
            if rng.random() < 0.4:
                b = thin_tracks(b, rng)
            B.ut_tuning_set(**tun) if tun else B.ut_tuning_set(None)
            h_ref, t_ref = oracle.run_batch(b, geom, p)
            T = b.n_velo_total
            T1, Tp = max(T, 1), (max(T, 1) + 63) // 64 * 64
            raw_h = B.to_host_pinned(np.concatenate([b.raw, np.zeros(32, np.uint8)]))
            bo_h, vo_h = B.to_host_pinned(b.bank_offsets.view(np.int32)), B.to_host_pinned(b.velo_offsets.view(np.int32))
            velo_blk = B.host_tensor(4 * Tp, torch.float32)
            velo_h = [velo_blk[r * Tp:r * Tp + T] for r in range(4)]
            for dst, src in zip(velo_h, (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty)):
                dst.numpy()[:] = src
            blocks = [raw_h, bo_h, vo_h, velo_blk]
            if one:                                   # the track SoA as one [7][T] block
                blk = B.host_tensor(7 * T1 + 32, torch.int32)
                blk.fill_(-7)
                out_h = {"hit_idx": blk[0:4 * T1], "n_hits": blk[4 * T1:5 * T1], "qop": blk[5 * T1:6 * T1].view(torch.float32),
                         "chi2": blk[6 * T1:7 * T1].view(torch.float32)}
                blocks.append(blk)
            else:
                blk, idx = B.host_tensor(3 * Tp, torch.int32), B.host_tensor(4 * T1, torch.int32)
                out_h = {"hit_idx": idx, "n_hits": blk[0:T1], "qop": blk[Tp:Tp + T1].view(torch.float32),
                         "chi2": blk[2 * Tp:2 * Tp + T1].view(torch.float32)}
                blocks += [blk, idx]
            out_h["status"], out_h["n_hits_total"] = B.host_tensor(2, torch.int32), B.host_tensor(1, torch.int32)
            blocks += [out_h["status"], out_h["n_hits_total"]]
            pipe = B.Pipeline(gpu.geom, ne, int(b.raw.size) + 32, b.hit_capacity, T1)
            try:
                for _ in range(3 if c == 4 else 2):
                    out_h["status"].fill_(-1)
                    out_h["n_hits"].fill_(-9)
                    pipe.run_host(raw_h, int(b.raw.size), bo_h, velo_h, b.velo_z, vo_h, T, ne, B.make_config(p), out_h)
                    torch.cuda.synchronize()
                    what = (c, ne, tun, one)
                    assert int(out_h["n_hits_total"][0]) == h_ref.n_hits and out_h["status"].tolist() == [0, 0], what
                    if T:
                        assert np.array_equal(out_h["hit_idx"].numpy().reshape(4, T1)[:, :T], t_ref.hit_idx), what
                    assert np.array_equal(out_h["n_hits"].numpy()[:T], t_ref.n_hits), what
                    assert np.array_equal(out_h["chi2"].numpy()[:T].view(np.uint32), t_ref.chi2.view(np.uint32)), what
                    assert np.array_equal(out_h["qop"].numpy()[:T].view(np.uint32), t_ref.qop.view(np.uint32)), what
                    if one:
                        assert np.all(blk.numpy()[7 * T1:] == -7), what
            finally:
                pipe.destroy()
                for t_ in blocks:
                    B.host_free(t_)
    finally:
        B.ut_tuning_set(None)
