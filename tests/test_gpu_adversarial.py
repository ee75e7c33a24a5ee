"""-m gpu: adversarial parity.  The hand-built cases of tests/adversarial_cases.py (exact window / y / seed / chi2
boundaries and one ulp either side, exact |d| ties at the cap, bit-identical chi2 from different lanes) run through
the CUDA path on both window-search paths and must equal the oracle bit for bit AND decide as the construction
predicts; malformed banks (A22) on both sides; capacity overflow followed by tracking; NaN VELO states;
canaries around every output (the pool has no compute-sanitizer); CUDA-graph replay; two host threads."""
import dataclasses
import threading

import numpy as np
import pytest

import adversarial_cases as AC
import oracle
import synth
from synth.events import assemble_batch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu(geom):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from gpu_helpers import GpuRunner
    return GpuRunner(geom)


@pytest.fixture(params=["view", "restage", "global", "split4"])
def run(request, gpu):
    """run(geom, batch, params): GPU == oracle bit for bit, returns the oracle's (hits, tracks).  Every data path
    of compass_track: per-sector buckets in shared memory taken from the decode's per-sector view (bulk copies) or
    re-bucketed by the kernel (container without the view), the search on global memory (the path of events that
    do not fit the staging), and four CTAs sharing one event's tracks."""
    from gpu_helpers import compare_decode
    gpu.B.ut_tuning_set(compass_hit_stage=0 if request.param == "global" else -1,
                        compass_split=4 if request.param == "split4" else -1)
    gpu.sector_view = request.param != "restage"

    def run_both(geom, b, p):
        h_ref, t_ref = oracle.run_batch(b, geom, p)
        hits, trk = gpu.run(b, p)
        got, off, st = gpu.hits_numpy(hits, b.n_events)
        compare_decode(h_ref, got, off, st)
        assert trk["status"] == 0
        assert np.array_equal(trk["hit_idx"], t_ref.hit_idx), (trk["hit_idx"], t_ref.hit_idx)
        assert np.array_equal(trk["n_hits"], t_ref.n_hits)
        assert np.array_equal(trk["chi2"].view(np.uint32), t_ref.chi2.view(np.uint32))
        assert np.array_equal(trk["qop"].view(np.uint32), t_ref.qop.view(np.uint32))
        return h_ref, t_ref

    yield run_both
    gpu.B.ut_tuning_set(None)
    gpu.sector_view = True


@pytest.mark.parametrize("layer", [0, 1, 2, 3])
def test_window_edge_exact(run, geom, layer):
    AC.case_window_edge_exact(run, geom, layer)


@pytest.mark.parametrize("layer", [0, 1, 2, 3])
def test_y_edge_exact(run, geom, layer):
    AC.case_y_edge_exact(run, geom, layer)


def test_seed_cut_edges(run, geom):
    AC.case_seed_cut_edges(run, geom)


def test_chi2_cut_edge(run, geom):
    AC.case_chi2_cut_edge(run, geom)


def test_abs_d_ties_at_the_cap(run, geom):
    AC.case_abs_d_ties_at_the_cap(run, geom)


def test_exact_chi2_ties_across_lanes(run, geom):
    AC.case_exact_chi2_ties_across_lanes(run, geom)


# ---------------------------------------------------------------------------------------------------
# malformed input on both sides (A22), capacity overflow followed by tracking, NaN VELO state
# ---------------------------------------------------------------------------------------------------
def test_malformed_banks(gpu, geom):
    from gpu_helpers import compare_decode
    import malformed
    raw, offs, want, _ = malformed.misaligned_tail(geom)
    ref = oracle.decode(raw, offs, 1, geom)
    hits = gpu.decode(raw, offs, 1, (raw.size - 6 * 896) // 2)
    got, off, st = gpu.hits_numpy(hits, 1)
    compare_decode(ref, got, off, st)
    assert st == gpu.B.UT_STATUS_BAD_BANK_SIZE and sorted(got["id"].astype(np.int64).tolist()) == want
    raw, offs, want2 = malformed.foreign_bank(geom)
    ref = oracle.decode(raw, offs, 2, geom)
    hits = gpu.decode(raw, offs, 2, (raw.size - 6 * 2 * 896) // 2)
    got, off, st = gpu.hits_numpy(hits, 2)
    compare_decode(ref, got, off, st)
    assert st == gpu.B.UT_STATUS_BAD_BANK_SIZE
    assert sorted(got["id"][int(off[64]):].astype(np.int64).tolist()) == want2[1]


def test_compass_after_capacity_overflow(gpu, wl):
    """ut_decode with a too-small container skips the overflowing events (UT_STATUS_CAPACITY, offsets exact);
    compass_track on that container must not read past `capacity`: those events get "no tracklet" and the status
    bit, the events that fit equal the oracle.  Same through ut_pipeline_run_host."""
    import torch
    from gpu_helpers import guarded_hits, check_guards
    geom, b, p = wl(2, 24)
    h_ref, t_ref = oracle.run_batch(b, geom, p)
    ev_end = h_ref.hit_offsets[64::64].astype(np.int64)
    cap = int(ev_end[15]) + 7                                             # events 0..15 fit, 16.. do not
    B = gpu.B
    hits, guards = guarded_hits(B, cap, b.n_events, gpu.geom)
    B.ut_decode(B.to_device_raw(b.raw), B.to_device_u32(b.bank_offsets), b.n_events, gpu.geom, hits)
    torch.cuda.synchronize()
    assert int(hits.status.item()) == B.UT_STATUS_CAPACITY
    assert np.array_equal(hits.hit_offsets.cpu().numpy().view(np.uint32), h_ref.hit_offsets)
    trk = gpu.compass(hits, b, p)
    check_guards(guards)
    assert trk["status"] == B.UT_STATUS_CAPACITY
    fit = np.repeat(np.arange(b.n_events) < 16, np.diff(b.velo_offsets.astype(np.int64)))
    assert np.array_equal(trk["hit_idx"][:, fit], t_ref.hit_idx[:, fit]) and (t_ref.n_hits[fit] > 0).sum() > 500
    assert np.array_equal(trk["chi2"][fit].view(np.uint32), t_ref.chi2[fit].view(np.uint32))
    assert np.all(trk["n_hits"][~fit] == 0) and np.all(trk["hit_idx"][:, ~fit] == -1)
    # the host pipeline with an arena that is too small for the hits
    T = b.n_velo_total
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    out_h = {"hit_idx": torch.full((4 * T,), -7, dtype=torch.int32).pin_memory(),
             "n_hits": torch.full((T,), -7, dtype=torch.int32).pin_memory(),
             "qop": torch.zeros(T, dtype=torch.float32).pin_memory(), "chi2": torch.zeros(T, dtype=torch.float32).pin_memory(),
             "status": torch.zeros(2, dtype=torch.int32).pin_memory(), "n_hits_total": torch.zeros(1, dtype=torch.int32).pin_memory()}
    pipe = B.Pipeline(gpu.geom, b.n_events, int(b.raw.size) + 32, cap, T)
    pipe.run_host(pin(np.concatenate([b.raw, np.zeros(32, np.uint8)])), int(b.raw.size), pin(b.bank_offsets.view(np.int32)),
                  [pin(v) for v in (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty)], b.velo_z, pin(b.velo_offsets.view(np.int32)),
                  T, b.n_events, B.make_config(p), out_h)
    torch.cuda.synchronize()
    assert out_h["status"].tolist() == [B.UT_STATUS_CAPACITY, B.UT_STATUS_CAPACITY]
    assert int(out_h["n_hits_total"][0]) == h_ref.n_hits
    assert np.array_equal(out_h["hit_idx"].numpy().reshape(4, T)[:, fit], t_ref.hit_idx[:, fit])
    assert np.all(out_h["n_hits"].numpy()[~fit] == 0)
    pipe.destroy()


def test_nan_velo_state(gpu, wl):
    """A NaN VELO state must not disturb the radius ordering of its event: every other track of the batch equals
    the oracle, the NaN track gets no tracklet, and nothing is written outside the track arrays."""
    import torch
    from gpu_helpers import guarded_tracks, check_guards
    geom, b, p = wl(2, 6)
    vo = b.velo_offsets.astype(np.int64)
    bad = [int(vo[1]) + 3, int(vo[1]) + 40, int(vo[4])]
    assert vo[2] - vo[1] > 48
    vx = b.velo_x.copy(); vy = b.velo_y.copy(); vtx = b.velo_tx.copy()
    vx[bad[0]] = np.nan; vy[bad[1]] = np.nan; vtx[bad[2]] = np.nan
    b2 = dataclasses.replace(b, velo_x=vx, velo_y=vy, velo_tx=vtx)
    h_ref, t_ref = oracle.run_batch(b2, geom, p)
    assert np.all(t_ref.n_hits[bad] == 0)
    B = gpu.B
    hits = gpu.decode(b2.raw, b2.bank_offsets, b2.n_events, b2.hit_capacity)
    velo = B.VeloStates(b2.velo_x, b2.velo_y, b2.velo_tx, b2.velo_ty, b2.velo_z)
    tracks, guards = guarded_tracks(B, b2.n_velo_total)
    B.compass_track(hits, hits.hit_offsets, velo, B.to_device_u32(b2.velo_offsets), b2.n_events, B.make_config(p), tracks)
    torch.cuda.synchronize()
    check_guards(guards)
    idx, n, qop, chi2 = tracks.numpy()
    assert np.array_equal(idx, t_ref.hit_idx) and np.array_equal(n, t_ref.n_hits)
    assert np.array_equal(chi2.view(np.uint32), t_ref.chi2.view(np.uint32))


# ---------------------------------------------------------------------------------------------------
# guard bands around every output, CUDA-graph replay, two host threads
# ---------------------------------------------------------------------------------------------------
def _guarded_run(gpu, geom, b, p, capacity=None):
    import torch
    from gpu_helpers import guarded_hits, guarded_tracks, guarded_compact, check_guards, compare_decode
    B = gpu.B
    cap = b.hit_capacity if capacity is None else capacity
    hits, g1 = guarded_hits(B, cap, b.n_events, gpu.geom)
    tracks, g2 = guarded_tracks(B, b.n_velo_total)
    compact, g3 = guarded_compact(B, b.n_velo_total, b.n_velo_total, b.n_events)
    velo = B.VeloStates(b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z)
    vo = B.to_device_u32(b.velo_offsets)
    B.ut_decode(B.to_device_raw(b.raw), B.to_device_u32(b.bank_offsets), b.n_events, gpu.geom, hits)
    B.compass_track(hits, hits.hit_offsets, velo, vo, b.n_events, B.make_config(p), tracks)
    B.compass_consolidate(tracks, vo, b.n_events, compact)
    torch.cuda.synchronize()
    check_guards(g1 + g2 + g3)
    return hits, tracks, compact


@pytest.mark.parametrize("case", ["config2", "config4", "generic_paths", "capacity", "edge_events"])
def test_guard_bands(gpu, geom, wl, case):
    """4 KB of canaries in front of and behind every output array of ut_decode, compass_track and
    compass_consolidate (exactly-sized arrays: a store one element past the end lands in a canary)."""
    from gpu_helpers import compare_decode
    B = gpu.B
    cap = None
    if case == "config2":
        g, b, p = wl(2)
    elif case == "config4":
        g, b, p = wl(4, 12)
    elif case == "generic_paths":
        g, b, p = wl(2, 12)
        B.ut_tuning_set(decode_sort_buf=32, decode_raw_stage_bytes=4096, compass_hit_stage=512, decode_hit_stage=0)
    elif case == "capacity":
        g, b, p = wl(2, 12)
        cap = int(oracle.decode(b.raw, b.bank_offsets, b.n_events, g, b.hit_capacity).hit_offsets[64 * 7]) + 1
    else:
        from synth.events import EventModel, generate_event
        evs = [generate_event(g_, m, 9, k) for k, (g_, m) in enumerate(
            [(geom, EventModel(fixed_tracks=0, noise_mean=0.0)), (geom, EventModel(fixed_tracks=3, noise_mean=40000.0)),
             (geom, EventModel(fixed_tracks=9, noise_mean=0.0, efficiency=1.0)), (geom, EventModel(fixed_tracks=300, noise_mean=10.0))])]
        g, b, p = geom, assemble_batch(geom, evs), synth.make_compass_params()
    try:
        hits, tracks, compact = _guarded_run(gpu, g, b, p, cap)
    finally:
        B.ut_tuning_set(None)
    h_ref = oracle.decode(b.raw, b.bank_offsets, b.n_events, g, b.hit_capacity if cap is None else cap)
    assert np.array_equal(hits.hit_offsets.cpu().numpy().view(np.uint32), h_ref.hit_offsets)
    if cap is None:
        got, off, st = gpu.hits_numpy(hits, b.n_events)
        compare_decode(h_ref, got, off, st)
        t_ref = oracle.compass(h_ref, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events, g, p)
        idx, n, qop, chi2 = tracks.numpy()
        assert np.array_equal(idx, t_ref.hit_idx) and np.array_equal(chi2.view(np.uint32), t_ref.chi2.view(np.uint32))
        c_ref = oracle.consolidate(t_ref.hit_idx, t_ref.n_hits, t_ref.qop, t_ref.chi2, b.velo_offsets, b.n_events)
        c = compact.numpy(b.n_events)
        assert np.array_equal(c["track_offsets"], c_ref.track_offsets) and np.array_equal(c["velo_index"], c_ref.velo_index)


def test_cuda_graph_replay(gpu, wl):
    """ut_decode + compass_track + compass_consolidate captured once in a CUDA graph and replayed on new inputs
    copied into the same buffers (include/ut_compass.h: "CUDA-graph capturable": no sync, no allocation, and the
    workspaces re-arm themselves on the device)."""
    import torch
    from gpu_helpers import compare_decode
    B = gpu.B
    geom, b0, p = wl(2, 40)
    _, b1, _ = wl(3, 40)
    batches = [b0, b1, b0]
    cap = max(x.hit_capacity for x in batches)
    T = max(x.n_velo_total for x in batches)
    raw_d = torch.zeros(max(x.raw.size for x in batches) + 64, dtype=torch.uint8, device="cuda")
    bo_d = torch.zeros(40 * 896 + 1, dtype=torch.int32, device="cuda")
    vo_d = torch.zeros(41, dtype=torch.int32, device="cuda")
    vel = [torch.zeros(T, dtype=torch.float32, device="cuda") for _ in range(4)]
    velo = B.VeloStates(*vel, b0.velo_z)
    hits = B.Hits(cap, 40, gpu.geom)
    tracks = B.Tracks(T)
    compact = B.CompactTracks(T, T, 40)
    cfg = B.make_config(p)

    def load(x):
        raw_d.zero_()
        raw_d[:x.raw.size] = torch.from_numpy(x.raw)
        bo_d.copy_(torch.from_numpy(x.bank_offsets.view(np.int32)))
        vo_d.copy_(torch.from_numpy(x.velo_offsets.view(np.int32)))
        for t, a in zip(vel, (x.velo_x, x.velo_y, x.velo_tx, x.velo_ty)):
            t.zero_()
            t[:a.size] = torch.from_numpy(a)

    def path():
        B.ut_decode(raw_d, bo_d, 40, gpu.geom, hits)
        B.compass_track(hits, hits.hit_offsets, velo, vo_d, 40, cfg, tracks)
        B.compass_consolidate(tracks, vo_d, 40, compact)

    load(b0)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        path()                                       # per-device set-up happens outside the capture
    side.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        path()
    for x in batches:
        load(x)
        for t in (hits.x_at_y0, hits.id, hits.hit_offsets, tracks.hit_idx, tracks.n_hits, tracks.chi2, compact.track_offsets):
            t.fill_(-3)
        hits.status.zero_(); tracks.status.zero_(); compact.status.zero_()
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        h_ref, t_ref = oracle.run_batch(x, geom, p)
        got, off, st = gpu.hits_numpy(hits, 40)
        compare_decode(h_ref, got, off, st)
        n = x.n_velo_total
        # the row stride of hit_idx is velo_offsets[n_events] of THIS batch (read on the device)
        idx = tracks.hit_idx[:4 * n].cpu().numpy().reshape(4, n)
        assert np.array_equal(idx, t_ref.hit_idx)
        assert np.array_equal(tracks.chi2[:n].cpu().numpy().view(np.uint32), t_ref.chi2.view(np.uint32))
        c_ref = oracle.consolidate(t_ref.hit_idx, t_ref.n_hits, t_ref.qop, t_ref.chi2, x.velo_offsets, 40)
        assert np.array_equal(compact.track_offsets.cpu().numpy().view(np.uint32), c_ref.track_offsets)


def test_back_to_back_calls_reuse_one_container(gpu, wl):
    """ut_decode and compass_track issued back to back on one stream, 40 times, alternating between batches of
    different sizes in the SAME container: compass_track is launched with programmatic stream serialization behind
    ut_decode (its CTAs may be resident before the decode completes), and nothing of the previous batch may leak
    into the next -- hits, offsets and tracks equal the oracle's every time."""
    import torch
    B = gpu.B
    work = [wl(3, 1000), wl(2, 100), wl(3, 333)]
    refs = [oracle.run_batch(b, g, p) for g, b, p in work]
    cap = max(b.hit_capacity for _, b, _ in work)
    hits = B.Hits(cap, 1000, gpu.geom)
    dev = [(B.to_device_raw(b.raw), B.to_device_u32(b.bank_offsets),
            B.VeloStates(b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z), B.to_device_u32(b.velo_offsets),
            B.Tracks(b.n_velo_total), B.make_config(p)) for _, b, p in work]
    ng = gpu.tables.n_groups
    for it in range(40):
        k = it % len(work)
        b = work[k][1]
        raw, bo, velo, vo, tracks, cfg = dev[k]
        B.ut_decode(raw, bo, b.n_events, gpu.geom, hits)
        B.compass_track(hits, hits.hit_offsets, velo, vo, b.n_events, cfg, tracks)
        torch.cuda.synchronize()
        h_ref, t_ref = refs[k]
        n = h_ref.n_hits
        assert np.array_equal(hits.hit_offsets[:b.n_events * ng + 1].cpu().numpy().view(np.uint32), h_ref.hit_offsets)
        assert np.array_equal(hits.x_at_y0[:n].cpu().numpy().view(np.uint32), h_ref.x_at_y0[:n].view(np.uint32))
        assert np.array_equal(hits.id[:n].cpu().numpy().view(np.uint32), h_ref.id[:n])
        idx, nh, qop, chi2 = tracks.numpy()
        assert np.array_equal(idx, t_ref.hit_idx) and np.array_equal(nh, t_ref.n_hits)
        assert np.array_equal(chi2.view(np.uint32), t_ref.chi2.view(np.uint32))
        assert np.array_equal(qop.view(np.uint32), t_ref.qop.view(np.uint32))
        assert int(tracks.status[0].item()) == 0


def test_two_compass_calls_share_one_container(gpu, wl):
    """DESIGN.md A21: the work ticket of compass_track lives in the OUTPUT (ut_tracks.status), so two calls that read
    the same hit container with different configs and outputs may run at the same time on two streams."""
    import dataclasses
    import torch
    from gpu_helpers import compare_tracks
    B = gpu.B
    g, b, p = wl(3, 200)
    p2 = dataclasses.replace(p, min_hits=4, max_candidates_per_layer=8)
    h_ref, t1 = oracle.run_batch(b, g, p)
    _, t2 = oracle.run_batch(b, g, p2)
    hits = gpu.decode(b.raw, b.bank_offsets, b.n_events, b.hit_capacity)
    velo = B.VeloStates(b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z)
    vo = B.to_device_u32(b.velo_offsets)
    tr = [B.Tracks(b.n_velo_total), B.Tracks(b.n_velo_total)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    for _ in range(5):
        for k, cfg in enumerate((p, p2)):
            B.compass_track(hits, hits.hit_offsets, velo, vo, b.n_events, B.make_config(cfg), tr[k], stream=streams[k])
    torch.cuda.synchronize()
    for k, ref in enumerate((t1, t2)):
        idx, nh, qop, chi2 = tr[k].numpy()
        got = dict(hit_idx=idx, n_hits=nh, qop=qop, chi2=chi2, status=int(tr[k].status[0].item()))
        n_diff, _ = compare_tracks(ref, got)
        assert n_diff == 0 and np.array_equal(chi2.view(np.uint32), ref.chi2.view(np.uint32))
        assert int(tr[k].status[0].item()) == 0


def test_two_host_threads(gpu, wl):
    """Two host threads, each with its own stream, container and outputs, call the library at the same time
    (per-device state is built under a lock; launch info and error text are thread-local)."""
    import torch
    from gpu_helpers import compare_decode
    B = gpu.B
    work = [wl(2, 60), wl(3, 60)]
    refs = [oracle.run_batch(b, g, p) for g, b, p in work]
    results, errors = [None, None], []

    def worker(k):
        try:
            g, b, p = work[k]
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                hits = B.Hits(b.hit_capacity, b.n_events, gpu.geom)
                raw_d, bo_d = B.to_device_raw(b.raw), B.to_device_u32(b.bank_offsets)
                velo = B.VeloStates(b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z)
                vo = B.to_device_u32(b.velo_offsets)
                tracks = B.Tracks(b.n_velo_total)
                cfg = B.make_config(p)
                s.synchronize()
                for _ in range(20):
                    B.ut_decode(raw_d, bo_d, b.n_events, gpu.geom, hits, stream=s)
                    B.compass_track(hits, hits.hit_offsets, velo, vo, b.n_events, cfg, tracks, stream=s)
                s.synchronize()
                results[k] = (gpu.hits_numpy(hits, b.n_events), tracks.numpy(), int(tracks.status[0].item()))
        except Exception as exc:                     # surfaced in the main thread
            errors.append(exc)

    ts = [threading.Thread(target=worker, args=(k,)) for k in range(2)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errors, errors
    for k in range(2):
        (got, off, st), (idx, n, qop, chi2), tst = results[k]
        compare_decode(refs[k][0], got, off, st)
        assert tst == 0 and np.array_equal(idx, refs[k][1].hit_idx)
        assert np.array_equal(chi2.view(np.uint32), refs[k][1].chi2.view(np.uint32))
