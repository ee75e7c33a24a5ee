"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element."""
import dataclasses

import numpy as np
import pytest

import oracle
import synth
from synth import geometry as G
from synth.events import EventModel, encode_event, generate_batch, assemble_batch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu(geom):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from gpu_helpers import GpuRunner
    return GpuRunner(geom)


def oracle_run(b, geom, p):
    return oracle.run_batch(b, geom, p)


def check_batch(gpu, geom, b, p):
    from gpu_helpers import compare_decode, compare_tracks
    h_ref, t_ref = oracle_run(b, geom, p)
    hits, trk = gpu.run(b, p)
    got, off, st = gpu.hits_numpy(hits, b.n_events)
    compare_decode(h_ref, got, off, st)
    n_diff, n_tie = compare_tracks(t_ref, trk)
    # identical fp32 arithmetic on both sides: even the flagged near-ties are expected to agree
    assert n_diff == 0
    assert np.array_equal(trk["chi2"].view(np.uint32), t_ref.chi2.view(np.uint32))
    assert np.array_equal(trk["qop"].view(np.uint32), t_ref.qop.view(np.uint32))
    return h_ref, t_ref


def test_config1(gpu, wl):
    geom, b, p = wl(1)
    h, t = check_batch(gpu, geom, b, p)
    assert (t.n_hits > 0).sum() >= 10


def test_config2(gpu, wl):
    geom, b, p = wl(2)
    check_batch(gpu, geom, b, p)


def check_sector_view(gpu, geom, b, hits, h_ref):
    """The per-sector view ut_decode writes beside the container (include/ut_compass.h): for every event and dense
    sector the hits of that sector, in container order, found by their ids in the oracle's container."""
    ne, ng, ns = b.n_events, geom.n_groups, geom.n_sectors
    stride = gpu.B.ut_sector_offsets_stride(gpu.geom)
    so = hits.sector_offsets.cpu().numpy().view(np.uint16).reshape(-1, stride)[:ne]
    sx = hits.x_by_sector.cpu().numpy()
    si = hits.idx_by_sector.cpu().numpy().view(np.uint16)
    ev0 = h_ref.hit_offsets[::ng].astype(np.int64)
    sec = geom.id_to_sector[h_ref.id[:h_ref.n_hits] >> 9].astype(np.int64)
    for e in range(ne):
        lo, hi = int(ev0[e]), int(ev0[e + 1])
        assert so[e, ns + 1] == 0xA5A5 and so[e, ns] == hi - lo and so[e, 0] == 0
        cnt = np.bincount(sec[lo:hi], minlength=ns)
        assert np.array_equal(np.diff(so[e, :ns + 1].astype(np.int64)), cnt)
        order = np.argsort(sec[lo:hi], kind="stable")              # sector-major, container order inside a sector
        assert np.array_equal(si[lo:hi], order.astype(np.uint16))
        assert np.array_equal(sx[lo:hi].view(np.uint32), h_ref.x_at_y0[lo:hi][order].view(np.uint32))


def test_sector_view_contents(gpu, wl):
    for c, n in ((2, 40), (4, 10)):
        geom, b, p = wl(c, n)
        h_ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
        hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
        check_sector_view(gpu, geom, b, hits, h_ref)


@pytest.mark.parametrize("tuning", [dict(), dict(decode_hit_stage=0), dict(decode_hit_stage=1024),
                                    dict(decode_block=64), dict(decode_block=512, decode_raw_stage_bytes=4096),
                                    dict(decode_hit_stage=0, decode_sort_buf=64, decode_block=96)],
                         ids=["cta", "warp_per_group", "stage_too_small", "block64", "block512_raw_global", "slices64"])
def test_decode_data_paths(gpu, wl, tuning):
    """Every way ut_decode can order an event gives the oracle's container and the same per-sector view: the CTA-wide
    order (thread per hit), the warp-per-group order (events that do not fit, UT_ORDER_Y), small and large CTAs, raw
    banks read from global memory.  Config 2 and config 4 events plus hand-built ties across sectors and chunks."""
    from gpu_helpers import compare_decode
    gpu.B.ut_tuning_set(**tuning) if tuning else gpu.B.ut_tuning_set(None)
    try:
        for c, n in ((2, 30), (4, 6)):
            geom, b, p = wl(c, n)
            h_ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
            hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
            got, off, st = gpu.hits_numpy(hits, b.n_events)
            compare_decode(h_ref, got, off, st)
            li = gpu.B.last_launch_info()
            if "decode_hit_stage" in tuning:
                assert li["decode_hit_stage"] == tuning["decode_hit_stage"]
            if tuning.get("decode_hit_stage", -1) != 1024 and tuning.get("decode_sort_buf", -1) != 64:
                check_sector_view(gpu, geom, b, hits, h_ref)     # (undersized buffers may leave an event without a view)
        # equal x in different rows of one column (X layer: same strip and frac), 70 copies of 5 strips: ties inside a
        # 32-hit chunk, across chunks and across sectors
        geom = gpu.tables
        k = np.arange(70)
        sec = G.dense_sector(0, 5, 0) + k % 14
        strip = 100 + k // 14
        rng = np.random.default_rng(3)
        perm = rng.permutation(k.size)
        b = assemble_batch(geom, [_one_event(geom, sec[perm], strip[perm], np.ones(k.size, int), rng.permutation(896))])
        h_ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
        hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
        got, off, st = gpu.hits_numpy(hits, b.n_events)
        compare_decode(h_ref, got, off, st)
    finally:
        gpu.B.ut_tuning_set(None)


@pytest.mark.parametrize("split", [1, 2, 4])
@pytest.mark.parametrize("view", [True, False])
def test_compass_data_paths(gpu, wl, view, split):
    """Same results with and without the decode's per-sector view, and with 1, 2 or 4 CTAs per event."""
    geom, b, p = wl(3, 120)
    gpu.sector_view = view
    gpu.B.ut_tuning_set(compass_split=split)
    try:
        check_batch(gpu, geom, b, p)
        li = gpu.B.last_launch_info()
        assert li["compass_view"] == int(view) and li["compass_split"] == split
    finally:
        gpu.sector_view = True
        gpu.B.ut_tuning_set(None)


def test_config3_subset(gpu, wl):
    geom, b, p = wl(3, 300)          # several waves of CTAs, ragged tail
    check_batch(gpu, geom, b, p)


def test_config4_subset(gpu, wl):
    geom, b, p = wl(4, 40)
    h, t = check_batch(gpu, geom, b, p)
    assert (t.cand_n > p.max_candidates_per_layer).any()      # the candidate cap path runs on the GPU too


def test_config3_full_size_bench_launch(gpu, wl):
    """BASELINE.json configs[2] at its full size, in the launch configuration bench.py times (defaults of the
    library for a 1000-event batch): every output element against the oracle."""
    geom, b, p = wl(3)
    assert b.n_events == 1000
    check_batch(gpu, geom, b, p)
    li = gpu.B.last_launch_info()
    assert li["kernels_launched"] == 1 and li["compass_grid"] >= 148
    assert li["compass_event_order"] >= 1000          # the events were handed out by descending track count ...
    gpu.B.ut_tuning_set(compass_event_order=0)       # ... and in batch order: the same tracks either way
    try:
        check_batch(gpu, geom, b, p)
        assert gpu.B.last_launch_info()["compass_event_order"] == 0
    finally:
        gpu.B.ut_tuning_set(None)


def test_config4_full_size(gpu, wl):
    """configs[3] at its full size (1000 events, ~8000 hits, C = 32)."""
    geom, b, p = wl(4)
    assert b.n_events == 1000
    h, t = check_batch(gpu, geom, b, p)
    assert (t.cand_n > p.max_candidates_per_layer).sum() > 1000


def test_compass_event_order_uneven_batch(gpu, wl):
    """The Compass kernels hand the events of a batch out by descending track count (a stable counting sort every CTA
    computes for itself), here the large-CTA kernel.  A batch of more events than SMs whose track counts differ wildly -- every 7th event
    without tracks, every 5th with a quarter of its tracks, the last event empty too: every track of every event still
    gets exactly the oracle's result."""
    geom, b, p = wl(4, 170)
    vo = b.velo_offsets.astype(np.int64)
    keep = []
    for e in range(b.n_events):
        n = int(vo[e + 1] - vo[e])
        k = 0 if (e % 7 == 3 or e == b.n_events - 1) else (n // 4 if e % 5 == 1 else n)
        keep.append(np.arange(vo[e], vo[e] + k))
    idx = np.concatenate(keep)
    vo_new = np.concatenate([[0], np.cumsum([len(k) for k in keep])]).astype(np.uint32)
    b2 = dataclasses.replace(b, velo_x=b.velo_x[idx], velo_y=b.velo_y[idx], velo_tx=b.velo_tx[idx], velo_ty=b.velo_ty[idx],
                             velo_offsets=vo_new, truth_hit_id=b.truth_hit_id[idx], truth_q=b.truth_q[idx],
                             truth_p=b.truth_p[idx])
    gpu.B.ut_tuning_set(compass_block=512)        # (leaves shared memory for the table: at the automatic block size the
    try:                                          #  launch prefers one more warp per CTA to the event order)
        check_batch(gpu, geom, b2, p)
        li = gpu.B.last_launch_info()
        assert li["compass_block"] == 512 and li["compass_split"] == 1 and li["compass_event_order"] >= b.n_events
    finally:
        gpu.B.ut_tuning_set(None)


def test_config5_first_1000_events_all_settings(gpu, wl):
    """configs[4]: the 18 sweep settings on the first 1000 events of the 10000-event stream (events are
    generated independently of the batch size, so these are the sweep's own first 1000 events)."""
    from gpu_helpers import compare_tracks
    from synth.configs import SWEEP_MIN_HITS, SWEEP_SCALE, SWEEP_CANDIDATES
    geom, b, _ = wl(5, 1000)
    hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
    h_ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    got, off, st = gpu.hits_numpy(hits, b.n_events)
    from gpu_helpers import compare_decode
    compare_decode(h_ref, got, off, st)
    for mh in SWEEP_MIN_HITS:
        for sc in SWEEP_SCALE:
            for C in SWEEP_CANDIDATES:
                p = synth.CONFIGS[5].compass_params(min_hits=mh, window_scale=sc, max_candidates_per_layer=C)
                t_ref = oracle.compass(h_ref, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets,
                                       b.n_events, geom, p)
                trk = gpu.compass(hits, b, p)
                n_diff, _ = compare_tracks(t_ref, trk)
                assert n_diff == 0, (mh, sc, C)
                assert np.array_equal(trk["chi2"].view(np.uint32), t_ref.chi2.view(np.uint32)), (mh, sc, C)


@pytest.mark.parametrize("min_hits", [3, 4])
@pytest.mark.parametrize("scale", [0.5, 1.0, 2.0])
@pytest.mark.parametrize("C", [8, 16, 32])
def test_config5_sweep_subset(gpu, wl, min_hits, scale, C):
    geom, b, _ = wl(5, 60)
    p = synth.CONFIGS[5].compass_params(min_hits=min_hits, window_scale=scale, max_candidates_per_layer=C)
    from gpu_helpers import compare_tracks
    if not hasattr(gpu, "_c5"):
        gpu._c5 = (gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity),
                   oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity))
    hits, h_ref = gpu._c5
    t_ref = oracle.compass(h_ref, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events,
                           geom, p)
    trk = gpu.compass(hits, b, p)
    n_diff, _ = compare_tracks(t_ref, trk)
    assert n_diff == 0


def test_small_candidate_caps(gpu, wl):
    geom, b, _ = wl(2, 30)
    from gpu_helpers import compare_tracks
    hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
    h_ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    for C in (1, 2, 3, 5):
        p = synth.make_compass_params(max_candidates_per_layer=C, window_scale=2.0)
        t_ref = oracle.compass(h_ref, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets,
                               b.n_events, geom, p)
        assert (t_ref.cand_n > C).any()
        n_diff, _ = compare_tracks(t_ref, gpu.compass(hits, b, p))
        assert n_diff == 0


def _one_event(geom, sector, strip, frac, order=None):
    n = len(sector)
    raw, offs = encode_event(geom, np.asarray(sector, dtype=np.int64), np.asarray(strip), np.asarray(frac),
                             np.zeros(n, int), order)
    return dict(raw=raw, bank_offs=offs, velo=tuple(np.zeros(0, np.float32) for _ in range(4)),
                truth_hit_id=np.zeros((0, 4), np.int64), q=np.zeros(0, np.int8), p=np.zeros(0), n_hits=n)


def test_decode_edge_cases(gpu, geom):
    from gpu_helpers import compare_decode
    rng = np.random.default_rng(5)
    s_full = G.dense_sector(2, 7, 6)
    strips = np.arange(511, -1, -1)
    sec1 = np.repeat(np.arange(14) + G.dense_sector(1, 0, 0), 512)     # all hits of an event in one group
    st1 = np.tile(np.arange(512), 14)
    perm = rng.permutation(sec1.size)
    events = [
        _one_event(geom, [], [], []),                                   # empty event
        _one_event(geom, np.full(512, s_full), strips, strips % 2),     # one 512-word bank, descending order
        _one_event(geom, sec1[perm], st1[perm], np.zeros(sec1.size, int), rng.permutation(896)),
        _one_event(geom, [], [], []),
        _one_event(geom, [5, 5, 9, 895, 0], [1, 2, 3, 511, 0], [0, 1, 0, 1, 0]),
    ]
    b = assemble_batch(geom, events)
    ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
    got, off, st = gpu.hits_numpy(hits, b.n_events)
    compare_decode(ref, got, off, st)
    # no events
    hits = gpu.decode(np.zeros(0, np.uint8), np.zeros(1, np.uint32), 0, 0)
    assert int(hits.hit_offsets[0].item()) == 0


def test_decode_stable_ties(gpu, geom):
    from gpu_helpers import compare_decode
    # X layers: identical strips in every row of a column -> 14-way exact ties, order = dense sector
    sec = np.concatenate([np.arange(14) + G.dense_sector(0, c, 0) for c in (3, 8)])
    sec = np.repeat(sec, 3)
    strip = np.tile([100, 7, 300], 28)
    rng = np.random.default_rng(1)
    perm = rng.permutation(sec.size)
    b = assemble_batch(geom, [_one_event(geom, sec[perm], strip[perm], np.ones(sec.size, int), rng.permutation(896))])
    ref = oracle.decode(b.raw, b.bank_offsets, 1, geom, b.hit_capacity)
    hits = gpu.decode(b.raw, b.bank_offsets, 1, b.hit_capacity)
    got, off, st = gpu.hits_numpy(hits, 1)
    compare_decode(ref, got, off, st)


def test_decode_error_status(gpu, geom):
    e = _one_event(geom, [5, 5, 9], [1, 2, 3], [0, 0, 0])
    raw, offs = e["raw"], e["bank_offs"].astype(np.uint32)

    def both(r, capacity=None):
        cap = 3 if capacity is None else capacity
        ref = oracle.decode(r, offs, 1, geom, cap)
        hits = gpu.decode(r, offs, 1, cap)
        got, off, st = gpu.hits_numpy(hits, 1)
        return ref, got, off, st

    bad = raw.copy(); bad[int(offs[0]):int(offs[0]) + 4] = np.frombuffer(np.uint32(15).tobytes(), np.uint8)
    ref, got, off, st = both(bad)
    assert st == ref.status == oracle.ST_UNKNOWN_SECTOR and np.array_equal(off, ref.hit_offsets)
    bad = raw.copy(); bad[int(offs[0]):int(offs[0]) + 4] = raw[int(offs[1]):int(offs[1]) + 4]
    ref, got, off, st = both(bad)
    assert st == ref.status == oracle.ST_DUPLICATE_SECTOR
    bad = raw.copy(); bad[int(offs[5]) + 4] = 7
    ref, got, off, st = both(bad)
    assert st == ref.status == oracle.ST_BAD_BANK_SIZE and np.array_equal(off, ref.hit_offsets)
    ref, got, off, st = both(raw, capacity=2)
    assert st == ref.status == oracle.ST_CAPACITY and np.array_equal(off, ref.hit_offsets)


def test_repeated_calls_reuse_workspace(gpu, wl):
    """The look-back workspace re-arms itself: same buffers, several calls, different batch sizes."""
    from gpu_helpers import compare_decode
    geom, b, p = wl(2)
    ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    B, torch = gpu.B, gpu.torch
    hits = B.Hits(b.hit_capacity, b.n_events, gpu.geom)
    raw_d, bo_d = B.to_device_raw(b.raw), B.to_device_u32(b.bank_offsets)
    for n in (100, 37, 100, 1, 100):
        hits.hit_offsets.zero_()
        B.ut_decode(raw_d, bo_d, n, gpu.geom, hits)
        torch.cuda.synchronize()
        off = hits.hit_offsets[:n * 64 + 1].cpu().numpy().view(np.uint32)
        assert np.array_equal(off, ref.hit_offsets[:n * 64 + 1])
    got, off, st = gpu.hits_numpy(hits, 100)
    compare_decode(ref, got, off, st)


def test_small_staging_takes_generic_paths(gpu, wl):
    """Force the events through the non-staged decode path and the global-memory Compass path (ut_tuning_set:
    the library reads its environment knobs once, so the launch shapes are set through the API)."""
    geom, b, p = wl(2, 12)
    gpu.B.ut_tuning_set(decode_sort_buf=32, decode_raw_stage_bytes=4096, compass_hit_stage=512, decode_hit_stage=0)
    try:
        t = gpu.B.ut_tuning_get()
        assert (t.decode_sort_buf, t.decode_raw_stage_bytes, t.compass_hit_stage, t.compass_block) == (32, 4096, 512, -1)
        check_batch(gpu, geom, b, p)
        li = gpu.B.last_launch_info()
        assert li["compass_hit_stage"] == 512
    finally:
        gpu.B.ut_tuning_set(None)


def test_tracks_empty_cases(gpu, geom):
    p = synth.make_compass_params()
    b = generate_batch(geom, EventModel(fixed_tracks=0, noise_mean=50.0), seed=2, n_events=3)
    hits, trk = gpu.run(b, p)
    assert trk["n_hits"].shape == (0,)
    b = generate_batch(geom, EventModel(fixed_tracks=5, noise_mean=0.0, efficiency=0.0), seed=2, n_events=2)
    hits, trk = gpu.run(b, p)
    assert np.all(trk["n_hits"] == 0) and np.all(trk["hit_idx"] == -1) and np.all(trk["qop"] == 0)


def test_invalid_arguments(gpu, wl):
    geom, b, p = wl(1)
    B = gpu.B
    hits = gpu.decode(b.raw, b.bank_offsets, 1, b.hit_capacity)
    velo = B.VeloStates(b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z)
    vo = B.to_device_u32(b.velo_offsets)
    tracks = B.Tracks(20)
    for bad in (dataclasses.replace(p, min_hits=2), dataclasses.replace(p, max_candidates_per_layer=0),
                dataclasses.replace(p, max_candidates_per_layer=33)):
        with pytest.raises(B.UTError):
            B.compass_track(hits, hits.hit_offsets, velo, vo, 1, B.make_config(bad), tracks)
    with pytest.raises(B.UTError):
        B.ut_decode(B.to_device_raw(b.raw), B.to_device_u32(b.bank_offsets), -1, gpu.geom, hits)


@pytest.mark.parametrize("zero_copy", [0, 1], ids=["staged", "zero_copy"])
@pytest.mark.parametrize("n_events", [1000, 37])
def test_host_pipeline_matches_oracle(gpu, wl, n_events, zero_copy):
    """ut_pipeline_run_host (HOST buffers in, HOST track SoA out; the call bench.py's e2e figure times).
    1000 events run as 4 overlapped chunks of 250 (the default is chunks of >= 500 events), 37 events as
    one call: both must equal the oracle element by element."""
    import torch
    gpu.B.ut_tuning_set(pipeline_chunk_events=250, pipeline_zero_copy=zero_copy)
    geom, b, p = wl(3, n_events)
    h_ref, t_ref = oracle_run(b, geom, p)
    B = gpu.B
    T = b.n_velo_total
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    raw_h = pin(np.concatenate([b.raw, np.zeros(32, np.uint8)]))
    bo_h, vo_h = pin(b.bank_offsets.view(np.int32)), pin(b.velo_offsets.view(np.int32))
    velo_h = [pin(v) for v in (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty)]
    out_h = {"hit_idx": torch.full((4 * T,), -7, dtype=torch.int32).pin_memory(),
             "n_hits": torch.full((T,), -7, dtype=torch.int32).pin_memory(),
             "qop": torch.zeros(T, dtype=torch.float32).pin_memory(),
             "chi2": torch.zeros(T, dtype=torch.float32).pin_memory(),
             "status": torch.full((2,), -1, dtype=torch.int32).pin_memory(),
             "n_hits_total": torch.zeros(1, dtype=torch.int32).pin_memory()}
    pipe = B.Pipeline(gpu.geom, b.n_events, int(b.raw.size) + 32, b.hit_capacity, T)
    for _ in range(2):                                   # second run: workspace and events are reused
        pipe.run_host(raw_h, int(b.raw.size), bo_h, velo_h, b.velo_z, vo_h, T, b.n_events, B.make_config(p), out_h)
        torch.cuda.synchronize()
        assert int(out_h["n_hits_total"][0]) == h_ref.n_hits
        assert out_h["status"].tolist() == [0, 0]
        assert np.array_equal(out_h["hit_idx"].numpy().reshape(4, T), t_ref.hit_idx)
        assert np.array_equal(out_h["n_hits"].numpy(), t_ref.n_hits)
        assert np.array_equal(out_h["chi2"].numpy().view(np.uint32), t_ref.chi2.view(np.uint32))
        assert np.array_equal(out_h["qop"].numpy().view(np.uint32), t_ref.qop.view(np.uint32))
        out_h["n_hits"].fill_(-7)
    pipe.destroy()
    gpu.B.ut_tuning_set(None)


@pytest.mark.parametrize("chunk,one_block", [(333, False), (120, False), (333, True), (250, True)])
def test_host_pipeline_library_buffers_and_timeline(gpu, wl, chunk, one_block):
    """ut_pipeline_run_host with buffers from ut_host_alloc: the four VELO arrays are rows of one allocation and so are
    n_hits / qop / chi2, which the call moves as one strided copy each (separate torch-pinned tensors, the test above,
    take one copy per array); one_block: the whole track SoA is one [7][T] host block (hit_idx rows, n_hits, qop, chi2
    back to back), which leaves by a single strided copy per chunk; 3 and 4 chunks of linearly falling size.  The result
    equals the oracle's, and ut_pipeline_timeline reports for every chunk: banks in <= decoded <= tracked <= tracks out."""
    import torch
    B = gpu.B
    B.ut_tuning_set(pipeline_chunk_events=chunk)
    geom, b, p = wl(3, 1000)
    h_ref, t_ref = oracle_run(b, geom, p)
    T = b.n_velo_total
    Tp = (T + 63) // 64 * 64
    raw_h = B.to_host_pinned(np.concatenate([b.raw, np.zeros(32, np.uint8)]))
    bo_h, vo_h = B.to_host_pinned(b.bank_offsets.view(np.int32)), B.to_host_pinned(b.velo_offsets.view(np.int32))
    velo_blk = B.host_tensor(4 * Tp, torch.float32)
    velo_h = [velo_blk[r * Tp:r * Tp + T] for r in range(4)]
    for dst, src in zip(velo_h, (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty)):
        dst.numpy()[:] = src
    if one_block:
        Tp = T
        res = B.host_tensor(7 * T + 64, torch.int32)                 # (+ a canary tail)
        res.fill_(-7)
        idx_h = res[0:4 * T]
        res3 = res[4 * T:]
    else:
        res = B.host_tensor(3 * Tp, torch.int32)
        res.fill_(-7)
        idx_h = B.host_tensor(4 * T, torch.int32)
        res3 = res
    out_h = {"hit_idx": idx_h, "n_hits": res3[0:T], "qop": res3[Tp:Tp + T].view(torch.float32),
             "chi2": res3[2 * Tp:2 * Tp + T].view(torch.float32), "status": B.host_tensor(2, torch.int32),
             "n_hits_total": B.host_tensor(1, torch.int32)}
    pipe = B.Pipeline(gpu.geom, b.n_events, int(b.raw.size) + 32, b.hit_capacity, T)
    try:
        for _ in range(2):
            pipe.run_host(raw_h, int(b.raw.size), bo_h, velo_h, b.velo_z, vo_h, T, b.n_events, B.make_config(p), out_h)
            torch.cuda.synchronize()
            assert int(out_h["n_hits_total"][0]) == h_ref.n_hits and out_h["status"].tolist() == [0, 0]
            assert np.array_equal(out_h["hit_idx"].numpy().reshape(4, T), t_ref.hit_idx)
            assert np.array_equal(out_h["n_hits"].numpy(), t_ref.n_hits)
            assert np.array_equal(out_h["chi2"].numpy().view(np.uint32), t_ref.chi2.view(np.uint32))
            assert np.array_equal(out_h["qop"].numpy().view(np.uint32), t_ref.qop.view(np.uint32))
            if one_block:
                assert np.all(res.numpy()[7 * T:] == -7)                                          # nothing past the block
            else:
                assert np.all(res.numpy()[T:Tp] == -7) and np.all(res.numpy()[Tp + T:2 * Tp] == -7)   # the pads between the rows
            tl = pipe.timeline()
            assert len(tl) == min(4, 1000 // chunk)
            for c in tl:
                assert 0 < c["banks_in"] <= c["decoded"] <= c["tracked"] <= c["tracks_out"] and 0 < c["velo_in"] <= c["tracked"]
            assert all(tl[k]["tracks_out"] <= tl[k + 1]["tracks_out"] for k in range(len(tl) - 1))
            out_h["n_hits"].fill_(-7)
    finally:
        pipe.destroy()
        B.ut_tuning_set(None)
        for t_ in (raw_h, bo_h, vo_h, velo_blk, res, out_h["status"], out_h["n_hits_total"]) + (() if one_block else (idx_h,)):
            B.host_free(t_)


def _consolidate_both(gpu, t_idx, t_n, t_qop, t_chi2, vo, n_events, capacity=None):
    """compass_consolidate on device copies of a dense track SoA vs oracle.consolidate."""
    import torch
    B = gpu.B
    T = int(vo[n_events])
    cap = T if capacity is None else capacity
    tr = B.Tracks(T)
    if T:
        tr.hit_idx[:4 * T] = torch.from_numpy(np.ascontiguousarray(t_idx, np.int32).reshape(-1)).cuda()
        tr.n_hits[:T] = torch.from_numpy(np.ascontiguousarray(t_n)).cuda()
        tr.qop[:T] = torch.from_numpy(np.ascontiguousarray(t_qop)).cuda()
        tr.chi2[:T] = torch.from_numpy(np.ascontiguousarray(t_chi2)).cuda()
    out = B.CompactTracks(cap, T, n_events)
    vo_d = B.to_device_u32(vo)
    for _ in range(2):                                   # the look-back workspace re-arms itself
        out.track_offsets.fill_(-1)
        B.compass_consolidate(tr, vo_d, n_events, out)
        torch.cuda.synchronize()
    got = out.numpy(n_events)
    ref = oracle.consolidate(t_idx, t_n, t_qop, t_chi2, vo, n_events, cap)
    assert got["status"] == ref.status
    assert np.array_equal(got["track_offsets"], ref.track_offsets)
    assert np.array_equal(got["velo_index"], ref.velo_index)
    assert np.array_equal(got["hit_idx"], ref.hit_idx) and np.array_equal(got["n_hits"], ref.n_hits)
    assert np.array_equal(got["qop"].view(np.uint32), ref.qop.view(np.uint32))
    assert np.array_equal(got["chi2"].view(np.uint32), ref.chi2.view(np.uint32))
    return ref


def test_consolidate_full_size(gpu, wl):
    """PAPER.md:460 on the Compass output of configs[2] and configs[3] at full size (147 / 586 tiles)."""
    for c in (3, 4):
        geom, b, p = wl(c)
        _, t = oracle_run(b, geom, p)
        ref = _consolidate_both(gpu, t.hit_idx, t.n_hits, t.qop, t.chi2, b.velo_offsets, b.n_events)
        assert 0 < len(ref.velo_index) < b.n_velo_total


def test_consolidate_edge_cases(gpu):
    rng = np.random.default_rng(3)

    def tracks(nt, p_keep):
        vo = np.concatenate([[0], np.cumsum(nt)]).astype(np.uint32)
        T = int(vo[-1])
        n = np.where(rng.random(T) < p_keep, rng.integers(3, 5, T), 0).astype(np.int32)
        idx = np.where(n[None, :] > 0, rng.integers(0, 10 ** 6, (4, T)), -1).astype(np.int32)
        return idx, n, rng.normal(0, 1, T).astype(np.float32), rng.random(T).astype(np.float32), vo

    for nt, pk in (([0, 0, 0], 0.5),                          # no VELO tracks at all
                   ([2048, 0, 0, 2048, 1], 0.5),              # boundaries exactly on tile edges, empty events
                   ([4096], 1.0), ([4095, 1], 0.0),           # everything / nothing kept
                   ([5000, 3, 0, 7000, 1, 1, 1], 0.7),
                   (rng.poisson(3, 3000), 0.9)):              # many events per tile
        a = tracks(np.asarray(nt), pk)
        _consolidate_both(gpu, *a, len(nt))
    a = tracks(np.asarray([3000, 3000]), 1.0)
    ref = _consolidate_both(gpu, *a, 2, capacity=4100)        # capacity: offsets stay exact, nothing past the end
    assert ref.status == 8


@pytest.mark.parametrize("shuffle_rows", [False, True], ids=["rows_sorted", "rows_shuffled"])
def test_non_uniform_geometry(shuffle_rows):
    """SURVEY.md 8(f) row 3 (layout part): decode + Compass parity on the staggered geometry of synth/variant.py
    (two pitches, narrow inner columns and rows, rows overlapping in y, per-sector z, 4096-entry id table,
    optionally unsorted rows) -- nothing in the kernels may depend on the regular 16 x 14 layout."""
    from gpu_helpers import GpuRunner
    from synth import variant as V
    geom = V.make_staggered_geometry(shuffle_rows=shuffle_rows)
    b = V.generate_batch_tables(geom, EventModel(mean_tracks=150.0, efficiency=0.97, noise_mean=1500.0), seed=22,
                                n_events=60)
    runner = GpuRunner(geom)
    for p in (synth.make_compass_params(), synth.make_compass_params(window_scale=2.0, max_candidates_per_layer=4),
              synth.make_compass_params(min_hits=4, max_candidates_per_layer=32)):
        h, t = check_batch(runner, geom, b, p)
        assert (t.n_hits == 4).sum() > 500


def test_both_directions_mode(gpu, wl):
    """SURVEY.md 8(f) row 4 (selection part): best of forward and backward seeds, configs[1] and a busy subset."""
    import dataclasses
    for c, n in ((2, None), (4, 30)):
        geom, b, p = wl(c, n)
        _, t = check_batch(gpu, geom, b, dataclasses.replace(p, both_directions=1))
        _, t0 = oracle_run(b, geom, p)
        assert (t.hit_idx != t0.hit_idx).any()
    B = gpu.B
    with pytest.raises(B.UTError):
        geom, b, p = wl(1)
        hits, _ = gpu.run(b, p)
        bad = B.make_config(p); bad.both_directions = 2
        B.compass_track(hits, hits.hit_offsets, B.VeloStates(b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z),
                        B.to_device_u32(b.velo_offsets), 1, bad, B.Tracks(20))


def test_compass_status_paths(gpu, geom):
    """Data-dependent errors of compass_track (include/ut_compass.h): an event of more than 65535 hits (A19), hit
    offsets that are not monotone, VELO offsets that run backwards.  The bad event gets "no tracklet" (or is
    skipped), the status word says why, and every other event still equals the oracle."""
    from synth.events import generate_event
    B, torch = gpu.B, gpu.torch
    small = EventModel(fixed_tracks=30, efficiency=0.97, noise_mean=300.0)
    huge = EventModel(fixed_tracks=30, efficiency=0.97, noise_mean=80000.0)
    b = assemble_batch(geom, [generate_event(geom, small, 5, 0), generate_event(geom, huge, 5, 1),
                              generate_event(geom, small, 5, 2)])
    p = synth.make_compass_params()
    h_ref, t_ref = oracle_run(b, geom, p)
    assert h_ref.hit_offsets[128] - h_ref.hit_offsets[64] > 65535
    hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)      # the decode has no such limit
    got, off, st = gpu.hits_numpy(hits, b.n_events)
    from gpu_helpers import compare_decode
    compare_decode(h_ref, got, off, st)
    trk = gpu.compass(hits, b, p)
    assert trk["status"] == B.UT_STATUS_EVENT_TOO_LARGE
    ev = np.repeat(np.arange(3), np.diff(b.velo_offsets.astype(np.int64)))
    ok = ev != 1
    assert np.all(trk["n_hits"][~ok] == 0) and np.all(trk["hit_idx"][:, ~ok] == -1) and np.all(trk["chi2"][~ok] == 0)
    assert np.array_equal(trk["hit_idx"][:, ok], t_ref.hit_idx[:, ok]) and (t_ref.n_hits[ok] > 0).sum() > 20
    assert np.array_equal(trk["chi2"][ok].view(np.uint32), t_ref.chi2[ok].view(np.uint32))

    # offsets of event 1 not monotone -> BAD_OFFSETS, that event empty, the others untouched
    b3 = assemble_batch(geom, [generate_event(geom, small, 6, k) for k in range(3)])
    h3, t3 = oracle_run(b3, geom, p)
    hits = gpu.decode(b3.raw, b3.bank_offsets, 3, b3.hit_capacity)
    o = hits.hit_offsets.clone()
    hits.hit_offsets[64 + 10], hits.hit_offsets[64 + 11] = o[64 + 11] + 5, o[64 + 10]
    trk = gpu.compass(hits, b3, p)
    ev = np.repeat(np.arange(3), np.diff(b3.velo_offsets.astype(np.int64)))
    assert trk["status"] == B.UT_STATUS_BAD_OFFSETS
    assert np.all(trk["n_hits"][ev == 1] == 0)
    assert np.array_equal(trk["hit_idx"][:, ev != 1], t3.hit_idx[:, ev != 1])

    # VELO offsets running backwards for event 1: nothing can be written for it, status says so
    hits.hit_offsets.copy_(o)
    vo = b3.velo_offsets.copy()
    vo[1], vo[2] = vo[2], vo[1]
    velo = B.VeloStates(b3.velo_x, b3.velo_y, b3.velo_tx, b3.velo_ty, b3.velo_z)
    tr = B.Tracks(b3.n_velo_total)
    tr.n_hits.fill_(-9)
    B.compass_track(hits, hits.hit_offsets, velo, B.to_device_u32(vo), 3, B.make_config(p), tr)
    torch.cuda.synchronize()
    assert int(tr.status[0].item()) & B.UT_STATUS_BAD_OFFSETS


def test_compass_bad_hit_id(gpu, geom):
    """A hit whose id names no sector of the geometry is ignored and reported (UT_STATUS_BAD_HIT_ID); events
    without such a hit are untouched."""
    from synth.events import generate_event
    B = gpu.B
    m = EventModel(fixed_tracks=30, efficiency=0.97, noise_mean=300.0)
    b = assemble_batch(geom, [generate_event(geom, m, 8, k) for k in range(3)])
    p = synth.make_compass_params()
    _, t_ref = oracle_run(b, geom, p)
    gpu.sector_view = False          # a container without the decode's per-sector view: compass_track reads the ids
    try:
        hits = gpu.decode(b.raw, b.bank_offsets, 3, b.hit_capacity)
    finally:
        gpu.sector_view = True
    k = int(hits.hit_offsets[64 + 3].item())                   # a hit of event 1
    hits.id[k] = (1023 << 9) | 5                                # raw sector id 1023 is not in the table
    trk = gpu.compass(hits, b, p)
    assert trk["status"] == B.UT_STATUS_BAD_HIT_ID
    ev = np.repeat(np.arange(3), np.diff(b.velo_offsets.astype(np.int64)))
    assert np.array_equal(trk["hit_idx"][:, ev != 1], t_ref.hit_idx[:, ev != 1])
    assert not (trk["hit_idx"][:, ev == 1] == k).any()


def test_consolidate_workspace_too_small(gpu):
    """n_velo_total above what the workspace was sized for: reported, nothing written, the next call still works."""
    B, torch = gpu.B, gpu.torch
    T = 5000
    tr = B.Tracks(T)
    tr.n_hits.fill_(3); tr.hit_idx.fill_(7); tr.qop.fill_(1.0); tr.chi2.fill_(2.0)
    vo = B.to_device_u32(np.array([0, 2000, T], np.uint32))
    out = B.CompactTracks(T, 1000, 2)                  # workspace for 1000 tracks only
    out.velo_index.fill_(-5)
    B.compass_consolidate(tr, vo, 2, out)
    torch.cuda.synchronize()
    assert int(out.status.item()) == B.UT_STATUS_BAD_OFFSETS and int(out.velo_index[0].item()) == -5
    out2 = B.CompactTracks(T, T, 2)
    B.compass_consolidate(tr, vo, 2, out2)
    torch.cuda.synchronize()
    assert out2.numpy(2)["track_offsets"].tolist() == [0, 2000, T] and int(out2.status.item()) == 0


def test_host_pipeline_empty_and_invalid(gpu, wl):
    import torch
    B = gpu.B
    geom, b, p = wl(1)
    pipe = B.Pipeline(gpu.geom, 4, 4096, 1024, 64)
    z = lambda dt, n=1: torch.zeros(n, dtype=dt).pin_memory()
    out_h = {"hit_idx": z(torch.int32, 4), "n_hits": z(torch.int32), "qop": z(torch.float32), "chi2": z(torch.float32),
             "status": torch.full((2,), -1, dtype=torch.int32).pin_memory(),
             "n_hits_total": torch.full((1,), -1, dtype=torch.int32).pin_memory()}
    velo_h = [z(torch.float32) for _ in range(4)]
    pipe.run_host(z(torch.uint8, 64), 0, z(torch.int32), velo_h, 770.0, z(torch.int32), 0, 0, B.make_config(p), out_h)
    torch.cuda.synchronize()
    assert out_h["status"].tolist() == [0, 0] and int(out_h["n_hits_total"][0]) == 0
    with pytest.raises(B.UTError):                      # more events than the arena was created for
        pipe.run_host(z(torch.uint8, 64), 0, z(torch.int32, 5 * 896 + 1), velo_h, 770.0, z(torch.int32, 6), 0, 5,
                      B.make_config(p), out_h)
    pipe.destroy()


def test_kick_lut(gpu):
    """SURVEY.md 8(f) row 4 (field table): per-track kappa and z_mag from the position-dependent kick table
    (ut_geometry.kick_*, A24), fused kernel and the two-kernel variant against the oracle bit for bit;
    a table smaller than the acceptance exercises the clamped look-ups."""
    import torch
    from gpu_helpers import GpuRunner
    from synth.events import generate_batch
    p = synth.make_compass_params()
    for kw in (dict(falloff=0.3, bow=120.0), dict(half_x=250.0, half_y=200.0, nx=7, ny=5)):
        g = synth.make_geometry()
        g.kick = synth.make_kick_lut(**kw)
        b = generate_batch(g, EventModel(mean_tracks=150.0, efficiency=0.97, noise_mean=1500.0), seed=41, n_events=40)
        runner = GpuRunner(g)
        h_ref, t_ref = check_batch(runner, g, b, p)
        # the table matters: the same events tracked with the constant kick give other q/p values
        t_const = oracle.compass(h_ref, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events,
                                 synth.make_geometry(), p)
        assert (t_const.qop != t_ref.qop).sum() > 1000
        # two-kernel variant with 5 sector groups
        B = runner.B
        hits = runner.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
        velo = B.VeloStates(b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z)
        vo = B.to_device_u32(b.velo_offsets)
        T = b.n_velo_total
        win = torch.empty(T * 40, dtype=torch.int16, device="cuda")
        st = torch.zeros(1, dtype=torch.int32, device="cuda")
        tr = B.Tracks(T)
        B.compass_search_windows(hits, hits.hit_offsets, velo, vo, b.n_events, B.make_config(p), 5, win, st)
        B.compass_tracklets_from_windows(hits, hits.hit_offsets, velo, vo, b.n_events, B.make_config(p), 5, win, tr)
        torch.cuda.synchronize()
        idx, n, qop, chi2 = tr.numpy()
        assert np.array_equal(idx, t_ref.hit_idx) and np.array_equal(qop.view(np.uint32), t_ref.qop.view(np.uint32))
        assert np.array_equal(chi2.view(np.uint32), t_ref.chi2.view(np.uint32))


@pytest.mark.parametrize("name", ["regular", "staggered", "staggered_shuffled_rows"])
def test_y_order(name):
    """SURVEY.md 8(f) row 3 (Y-sorted groups): ut_decode with UT_ORDER_Y against the
    oracle's order "y" bit for bit (container and per-sector view), and compass_track on that container -- per-sector
    view, re-bucketing, and the search on global memory by two binary searches over Y -- against the oracle's linear
    scan (mode 1) and its Y-window search (mode 3)."""
    from gpu_helpers import GpuRunner, compare_decode, compare_tracks
    from synth import variant as V
    if name == "regular":
        geom = synth.make_geometry()
        b = generate_batch(geom, EventModel(mean_tracks=150.0, efficiency=0.97, noise_mean=1500.0), 19, 40)
    else:
        geom = V.make_staggered_geometry(shuffle_rows=name.endswith("shuffled_rows"))
        b = V.generate_batch_tables(geom, EventModel(mean_tracks=150.0, efficiency=0.97, noise_mean=1500.0), seed=19, n_events=40)
    runner = GpuRunner(geom)
    runner.order = "y"
    h_ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity, order="y")
    args = (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events, geom)
    B = runner.B
    for p in (synth.make_compass_params(), synth.make_compass_params(min_hits=4, window_scale=2.0, max_candidates_per_layer=3)):
        t_ref = oracle.compass(h_ref, *args, p, mode=1)
        t3 = oracle.compass(h_ref, *args, p, mode=3)
        assert np.array_equal(t_ref.hit_idx, t3.hit_idx)
        for path in ("view", "restage", "global"):
            runner.sector_view = path != "restage"
            B.ut_tuning_set(compass_hit_stage=0 if path == "global" else -1)
            try:
                hits = runner.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
                got, off, st = runner.hits_numpy(hits, b.n_events)
                compare_decode(h_ref, got, off, st)
                trk = runner.compass(hits, b, p)
            finally:
                B.ut_tuning_set(None)
            n_diff, _ = compare_tracks(t_ref, trk)
            assert n_diff == 0, path
            assert np.array_equal(trk["chi2"].view(np.uint32), t_ref.chi2.view(np.uint32)), path
            assert np.array_equal(trk["qop"].view(np.uint32), t_ref.qop.view(np.uint32)), path
        assert (t_ref.n_hits > 0).sum() > 1000
    # the per-sector view of a Y-ordered container is the container itself, sector by sector in y order (where the
    # dense sector order is the y order; with shuffled rows ut_decode marks the view unusable and compass_track
    # re-buckets)
    runner.sector_view = True
    hits = runner.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
    n = h_ref.n_hits
    stride = B.ut_sector_offsets_stride(runner.geom)
    flags = hits.sector_offsets.cpu().numpy().view(np.uint16).reshape(-1, stride)[:b.n_events, geom.n_sectors + 1]
    if name.endswith("shuffled_rows"):
        assert np.all(flags == 0)
        return
    assert np.all(flags == 0xA5A5)
    assert np.array_equal(hits.x_by_sector[:n].cpu().numpy().view(np.uint32), h_ref.x_at_y0[:n].view(np.uint32))
    ev0 = np.repeat(h_ref.hit_offsets[::geom.n_groups][:-1].astype(np.int64), np.diff(h_ref.hit_offsets[::geom.n_groups].astype(np.int64)))
    assert np.array_equal(hits.idx_by_sector[:n].cpu().numpy().view(np.uint16).astype(np.int64), np.arange(n) - ev0)
    # the two-kernel variant searches x-sorted groups only
    with pytest.raises(B.UTError):
        import torch
        B.compass_search_windows(hits, hits.hit_offsets, B.VeloStates(b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z),
                                 B.to_device_u32(b.velo_offsets), b.n_events, B.make_config(synth.make_compass_params()), 3,
                                 torch.empty(b.n_velo_total * 24, dtype=torch.int16, device="cuda"),
                                 torch.zeros(1, dtype=torch.int32, device="cuda"))
