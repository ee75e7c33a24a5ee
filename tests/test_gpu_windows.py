"""-m gpu: the paper-literal two-kernel Compass (Fig. 7) against its oracle:
window ranges bit for bit (int16), tracklets bit for bit, for 1, 3 and 5 sector groups; with 5 the tracklets also
equal the fused compass_track."""
import numpy as np
import pytest

import oracle
import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu(geom):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from gpu_helpers import GpuRunner
    return GpuRunner(geom)


def run_two_kernel(gpu, hits, b, p, W):
    import torch
    B = gpu.B
    T = b.n_velo_total
    velo = B.VeloStates(b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z)
    vo = B.to_device_u32(b.velo_offsets)
    win = torch.full((max(T, 1) * 4 * 2 * W,), -9, dtype=torch.int16, device="cuda")
    st = torch.zeros(1, dtype=torch.int32, device="cuda")
    cfg = B.make_config(p)
    B.compass_search_windows(hits, hits.hit_offsets, velo, vo, b.n_events, cfg, W, win, st)
    tracks = B.Tracks(T)
    B.compass_tracklets_from_windows(hits, hits.hit_offsets, velo, vo, b.n_events, cfg, W, win, tracks)
    torch.cuda.synchronize()
    idx, n, qop, chi2 = tracks.numpy()
    return (win[:T * 8 * W].cpu().numpy().reshape(T, 4, 2 * W), int(st.item()) & 0xFFFFFFFF,
            dict(hit_idx=idx, n_hits=n, qop=qop, chi2=chi2, status=int(tracks.status[0].item()) & 0xFFFFFFFF))


def check(gpu, geom, b, p, fused_equal=True):
    h_ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
    args = (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events, geom)
    for W in (1, 3, 5):
        win_ref, st_ref = oracle.search_windows(h_ref, *args, p, W)
        t_ref = oracle.compass_from_windows(h_ref, win_ref, *args, p, W)
        win, st, trk = run_two_kernel(gpu, hits, b, p, W)
        assert st == st_ref and trk["status"] == 0
        assert np.array_equal(win, win_ref), np.argwhere(win != win_ref)[:5]
        assert np.array_equal(trk["hit_idx"], t_ref.hit_idx) and np.array_equal(trk["n_hits"], t_ref.n_hits)
        assert np.array_equal(trk["chi2"].view(np.uint32), t_ref.chi2.view(np.uint32))
        assert np.array_equal(trk["qop"].view(np.uint32), t_ref.qop.view(np.uint32))
        if W == 5 and fused_equal:
            fused = gpu.compass(hits, b, p)
            assert np.array_equal(trk["hit_idx"], fused["hit_idx"])
            assert np.array_equal(trk["chi2"].view(np.uint32), fused["chi2"].view(np.uint32))
    return t_ref


def test_config1_and_2(gpu, wl):
    for c, n in ((1, None), (2, 40)):
        geom, b, p = wl(c, n)
        t = check(gpu, geom, b, p)
        assert (t.n_hits > 0).sum() >= 10


def test_config4_subset_caps(gpu, wl):
    geom, b, p = wl(4, 8)
    t = check(gpu, geom, b, p)
    assert (t.cand_n > p.max_candidates_per_layer).any()


@pytest.mark.parametrize("min_hits,scale,C", [(4, 0.5, 8), (3, 2.0, 32), (3, 1.0, 1), (4, 1.0, 5)])
def test_settings(gpu, wl, min_hits, scale, C):
    geom, b, _ = wl(5, 30)
    p = synth.CONFIGS[5].compass_params(min_hits=min_hits, window_scale=scale, max_candidates_per_layer=C)
    check(gpu, geom, b, p)


def test_both_directions_and_variant_geometry(gpu, wl):
    import dataclasses
    from gpu_helpers import GpuRunner
    from synth import variant as V
    from synth.events import EventModel
    geom, b, p = wl(2, 20)
    check(gpu, geom, b, dataclasses.replace(p, both_directions=1))
    vg = V.make_staggered_geometry()
    vb = V.generate_batch_tables(vg, EventModel(mean_tracks=150.0, efficiency=0.97, noise_mean=1500.0), seed=23, n_events=20)
    check(GpuRunner(vg), vg, vb, synth.make_compass_params(), fused_equal=False)


def test_edge_events(gpu, geom):
    """No hits, no tracks, tracks pointing outside the acceptance, and an event shorts cannot index."""
    from synth.events import EventModel, generate_event, assemble_batch
    evs = [generate_event(geom, EventModel(fixed_tracks=0, noise_mean=50.0), 31, 0),
           generate_event(geom, EventModel(fixed_tracks=7, noise_mean=0.0, efficiency=0.0), 31, 1),
           generate_event(geom, EventModel(fixed_tracks=90, noise_mean=1200.0), 31, 2),
           generate_event(geom, EventModel(fixed_tracks=5, noise_mean=40000.0), 31, 3)]
    evs[2]["velo"] = tuple(v.copy() for v in evs[2]["velo"])
    evs[2]["velo"][0][:10] += np.float32(5000.0)              # ten tracks far outside every panel
    evs[2]["velo"][1][10:13] = np.float32(np.nan)
    b = assemble_batch(geom, evs)
    p = synth.make_compass_params()
    h_ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
    args = (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events, geom)
    for W in (3, 5):
        win_ref, st_ref = oracle.search_windows(h_ref, *args, p, W)
        t_ref = oracle.compass_from_windows(h_ref, win_ref, *args, p, W)
        win, st, trk = run_two_kernel(gpu, hits, b, p, W)
        assert st == st_ref == gpu.B.UT_STATUS_EVENT_TOO_LARGE
        assert np.array_equal(win, win_ref)
        assert np.array_equal(trk["hit_idx"], t_ref.hit_idx) and np.array_equal(trk["chi2"].view(np.uint32), t_ref.chi2.view(np.uint32))
        assert (t_ref.n_hits > 0).sum() > 30
