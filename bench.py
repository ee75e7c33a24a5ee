#!/usr/bin/env python
"""bench.py -- UT decode + Compass events/s on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A step = one pass of the whole hot path (ut_decode + compass_track) over one
synthetic batch (config 3: 1000 events, ~2000 hits and ~150 VELO tracks each, seed 3; rank r of N takes
events [r*1000, (r+1)*1000) of the same stream: weak scaling, no collective on the data path).
Timing: CUDA events on the launching stream around every step, L2 flushed (256 MiB memset) between
steps, barrier + synchronize on both sides of the timed region, max over ranks.
`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ut_decode_compass_events_per_s"
UNIT = "events/s"

NCU_COUNTERS = os.path.join(ROOT, "profiles", "ncu_counters.json")
CSRC = os.path.join(ROOT, "paper_2002_11529_b200", "csrc")


def csrc_hash() -> str:
    """sha256 over the kernel sources (names and contents): the key profiles/ncu_counters.json was captured at.
    (The GPU box has no .git, so the tree hash is computed from the files themselves.)"""
    import hashlib
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh")):
            h.update(name.encode())
            h.update(open(os.path.join(CSRC, name), "rb").read())
    return h.hexdigest()[:16]


def ncu_counters(workload: str):
    """Per-launch ncu counters (DRAM bytes, warp instructions) of the committed `ncu --set full` capture, or
    (None, reason) when the kernel sources changed since the capture: a stale figure is not reported."""
    try:
        doc = json.load(open(NCU_COUNTERS))
    except Exception as exc:
        return None, f"profiles/ncu_counters.json unreadable: {exc}"
    if doc.get("csrc_sha256_16") != csrc_hash():
        return None, (f"kernel sources changed since the capture (captured at {doc.get('csrc_sha256_16')} = commit "
                      f"{doc.get('commit')}, now {csrc_hash()}): re-run the ncu capture named in {doc.get('source')}")
    w = doc.get("workloads", {}).get(workload)
    if not w:
        return None, f"no ncu capture for workload {workload}"
    return dict(w, source=doc.get("source"), commit=doc.get("commit")), None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config (1-based); 3 is the metric's workload")
    ap.add_argument("--events", type=int, default=None, help="override the number of events per GPU")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (configs 1, 2, 4, 5)")
    ap.add_argument("--sweep", action="store_true", help="config 5: all 18 settings with efficiency / ghost rate")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------
# algorithmic bytes per launch: what the method must move once
# ---------------------------------------------------------------------------------------------------
def algorithmic_bytes(batch, geom, n_hits):
    ne, T = batch.n_events, batch.n_velo_total
    decode = batch.raw.size + 4 * (ne * geom.n_sectors + 1) + 28 * n_hits + 4 * (ne * geom.n_groups + 1)
    compass = 24 * n_hits + 4 * (ne * geom.n_groups + 1) + 4 * (ne + 1) + 16 * T + 28 * T
    e2e = decode + 4 * (ne + 1) + 16 * T + 28 * T
    return dict(decode=int(decode), compass=int(compass), e2e=int(e2e))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons while the GPU is under load (B200_PROFILING.md recipe)."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "10", "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None
        self.marks = []

    def mark(self):
        self.marks.append(time.time())

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.p.terminate()
        try:
            self.p.wait(timeout=2)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = []
        for line in open(self.f.name):
            parts = [x.strip() for x in line.split(",")]
            if len(parts) >= 9:
                try:
                    ts = time.mktime(time.strptime(parts[0].split(".")[0], "%Y/%m/%d %H:%M:%S")) + \
                        float("0." + parts[0].split(".")[1]) if "." in parts[0] else 0.0
                    rows.append((ts, float(parts[1]), float(parts[2]), parts[3], parts[5:9]))
                except ValueError:
                    pass
        os.unlink(self.f.name)
        lo, hi = (self.marks + [0, 0])[:2] if len(self.marks) >= 2 else (0, 1e18)
        sel = [r for r in rows if lo - 0.05 <= r[0] <= hi + 0.05] or rows
        if not sel:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in sel for i, v in enumerate(r[4]) if v.lower().startswith("active")})
        return {"sm_mhz": statistics.median(r[1] for r in sel), "sm_max_mhz": sel[0][2], "reasons": reasons,
                "samples": len(sel)}


def oracle_chunked(batch, geom, params, lo, hi, threads):
    """The oracle, as it stands, over disjoint event chunks on `threads` host threads (ctypes drops the GIL).
    Every thread decodes its chunk, waits for the others, then tracks it: returns the wall time of the decode
    phase, of the tracking phase and of both (SURVEY.md 8(d) "oracle timed beside it": decode-only,
    tracking-only, end to end)."""
    import oracle
    cuts = np.linspace(lo, hi, threads + 1).astype(int)
    ns = geom.n_sectors
    gate = threading.Barrier(threads)
    stamps = [0.0, 0.0, 0.0]

    def work(k, a, b):
        bo = batch.bank_offsets[a * ns:b * ns + 1]
        cap = max((int(bo[-1]) - int(bo[0]) - 6 * (b - a) * ns) // 2, 0)
        vo = batch.velo_offsets[a:b + 1]
        T = int(vo[-1]) - int(vo[0])
        out = oracle.Tracks(np.full((4, max(T, 1)), -1, np.int32), np.zeros(max(T, 1), np.int32),
                            np.zeros(max(T, 1), np.float32), np.zeros(max(T, 1), np.float32), None, None, None, None)
        sl = slice(int(vo[0]), int(vo[0]) + T)
        v = [np.ascontiguousarray(x[sl]) for x in (batch.velo_x, batch.velo_y, batch.velo_tx, batch.velo_ty)]
        vo0 = (vo - vo[0]).astype(np.uint32)
        gate.wait()
        if k == 0:
            stamps[0] = time.perf_counter()
        h = oracle.decode(batch.raw, bo, b - a, geom, cap) if b > a else None
        gate.wait()
        if k == 0:
            stamps[1] = time.perf_counter()
        if b > a and T > 0:
            oracle.compass_into(out, h, v[0], v[1], v[2], v[3], batch.velo_z, vo0, b - a, geom, params, 0, extras=False)
        gate.wait()
        if k == 0:
            stamps[2] = time.perf_counter()

    ts = [threading.Thread(target=work, args=(k, int(a), int(b))) for k, (a, b) in enumerate(zip(cuts[:-1], cuts[1:]))]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    return stamps[1] - stamps[0], stamps[2] - stamps[1], stamps[2] - stamps[0]


def time_oracle(batch, geom, params, threads, budget_s, max_reps=50):
    """events/s of the oracle on `threads` host threads over all events of `batch`: decode-only, tracking-only,
    end to end (sums over whole passes; at least one pass)."""
    n = batch.n_events
    reps, td, tc, tb = 0, 0.0, 0.0, 0.0
    while (tb < budget_s and reps < max_reps) or reps == 0:
        d, c, both = oracle_chunked(batch, geom, params, 0, n, threads)
        td, tc, tb, reps = td + d, tc + c, tb + both, reps + 1
    return {"events_per_s": n * reps / tb, "decode_only_events_per_s": n * reps / td,
            "tracking_only_events_per_s": n * reps / tc, "passes": reps, "wall_s": tb}


def cpu_baseline(batch, geom, params, budget_s=6.0):
    """The oracle as it stands on the GPU box's host cores: (i) one thread, (ii) all threads
    over disjoint event chunks; decode-only / tracking-only / end to end each."""
    import oracle
    oracle.build()
    cores = os.cpu_count() or 1
    n = batch.n_events
    oracle_chunked(batch, geom, params, 0, min(n, 4 * cores), min(cores, max(n, 1)))      # warm the library
    many = time_oracle(batch, geom, params, min(cores, max(n, 1)), budget_s)
    one = time_oracle(batch, geom, params, 1, budget_s / 2, max_reps=3)
    return {"value": many["events_per_s"], "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"all {n} events of the workload x {many['passes']} passes, oracle decode + compass on {cores} "
                      f"threads over disjoint event chunks ({many['wall_s']:.1f} s wall); one thread: {one['passes']} "
                      f"pass(es) over the same {n} events ({one['wall_s']:.1f} s)",
            "decode_only": many["decode_only_events_per_s"], "tracking_only": many["tracking_only_events_per_s"],
            "one_thread": {"value": one["events_per_s"], "decode_only": one["decode_only_events_per_s"],
                           "tracking_only": one["tracking_only_events_per_s"], "cores": 1}}


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle, as it stands, on the host cores: same metric, same config, the same
    events per step as the GPU arm (rank 0 alone runs it)."""
    if rank != 0:
        return
    import synth
    cfg = synth.CONFIGS[args.config]
    cores = os.cpu_count() or 1
    n = args.events or cfg.n_events
    geom, batch, params = synth.make_workload(args.config, n_events=n, workers=min(8, cores))
    import oracle
    oracle.build()
    threads = min(cores, max(n, 1))
    for _ in range(max(min(args.warmup, 3), 1)):
        oracle_chunked(batch, geom, params, 0, n, threads)
    td = tc = t = 0.0
    for _ in range(args.steps):
        d, c, both = oracle_chunked(batch, geom, params, 0, n, threads)
        td, tc, t = td + d, tc + c, t + both
    value = n * args.steps / t
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "impl": "reference",
            "config": {"workload": cfg.name, "events_per_step": n, "events_per_gpu": n,
                       "note": f"CPU oracle (oracle/ut_oracle.cpp) as it stands: all {n} events of the workload per "
                               f"step over disjoint event chunks on {threads} host threads"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"all {n} events of {cfg.name} per step, {args.steps} steps",
                             "decode_only": n * args.steps / td, "tracking_only": n * args.steps / tc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_sweep(args, local_rank):
    """--sweep: BASELINE.json configs[4] -- 10000 events of the config-2 distribution, Compass run with
    {min_hits 3, 4} x {window scale 0.5, 1, 2} x {max_candidates_per_layer 8, 16, 32}; per setting
    events/s (decode + Compass, L2 flushed between steps) with efficiency and ghost rate of the GPU
    tracklets against the generator truth (synth/truth.py)."""
    import synth
    from synth.configs import SWEEP_MIN_HITS, SWEEP_SCALE, SWEEP_CANDIDATES
    cfg = synth.CONFIGS[5]
    n_events = args.events or cfg.n_events
    geom_t, batch, _ = synth.make_workload(5, n_events=n_events, workers=min(8, os.cpu_count() or 1))
    import torch
    import __graft_entry__ as entry
    entry.build()
    torch.cuda.set_device(local_rank)
    from paper_2002_11529_b200 import binding as B
    dev = torch.device("cuda", local_rank)
    geom = B.ut_geometry_upload(geom_t)
    hits = B.Hits(batch.hit_capacity, batch.n_events, geom)
    raw_d, bo_d = B.to_device_raw(batch.raw), B.to_device_u32(batch.bank_offsets)
    velo = B.VeloStates(batch.velo_x, batch.velo_y, batch.velo_tx, batch.velo_ty, batch.velo_z)
    vo_d = B.to_device_u32(batch.velo_offsets)
    tracks = B.Tracks(batch.n_velo_total)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    steps = max(3, min(args.steps, 20))
    rows = []
    for mh in SWEEP_MIN_HITS:
        for sc in SWEEP_SCALE:
            for C in SWEEP_CANDIDATES:
                params = cfg.compass_params(min_hits=mh, window_scale=sc, max_candidates_per_layer=C)
                config = B.make_config(params)
                for _ in range(3):
                    flush.zero_()
                    B.ut_decode(raw_d, bo_d, batch.n_events, geom, hits)
                    B.compass_track(hits, hits.hit_offsets, velo, vo_d, batch.n_events, config, tracks)
                ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
                torch.cuda.synchronize()
                for k in range(steps):
                    flush.zero_()
                    ev[k][0].record(stream)
                    B.ut_decode(raw_d, bo_d, batch.n_events, geom, hits)
                    ev[k][1].record(stream)
                    B.compass_track(hits, hits.hit_offsets, velo, vo_d, batch.n_events, config, tracks)
                    ev[k][2].record(stream)
                torch.cuda.synchronize()
                md = statistics.mean(e[0].elapsed_time(e[1]) for e in ev)
                mc = statistics.mean(e[1].elapsed_time(e[2]) for e in ev)
                idx, nh, qop, _chi2 = tracks.numpy()
                n_hits = int(hits.hit_offsets[batch.n_events * geom.n_groups].item()) & 0xFFFFFFFF
                ids = hits.id[:n_hits].cpu().numpy().view(np.uint32)
                m = synth.physics_metrics(batch.truth_hit_id, batch.truth_q, ids, idx, nh, qop)
                rows.append({"min_hits": mh, "window_scale": sc, "max_candidates_per_layer": C,
                             "events_per_s": batch.n_events / (md + mc) * 1e3,
                             "tracking_only_events_per_s": batch.n_events / mc * 1e3,
                             "ms_decode": md, "ms_compass": mc, "efficiency": m["efficiency"],
                             "ghost_rate": m["ghost_rate"], "charge_ok": m["charge_ok"],
                             "four_hit_fraction": m["four_hit_fraction"], "n_tracklets": m["n_tracklets"],
                             "n_reconstructible": m["n_reconstructible"],
                             "status_word": (int(hits.status.item()) | int(tracks.status[0].item())) & 0xFFFFFFFF})
    base = next(r for r in rows if (r["min_hits"], r["window_scale"], r["max_candidates_per_layer"]) == (3, 1.0, 16))
    line = {"metric": METRIC, "value": base["events_per_s"], "unit": UNIT, "n_gpus": 1, "steps": steps, "warmup": 3,
            "ms_per_step": base["ms_decode"] + base["ms_compass"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg.name, "events_per_gpu": batch.n_events, "velo_tracks": batch.n_velo_total,
                       "l2": "flushed (256 MiB memset) between timed steps",
                       "note": "value = the (min_hits 3, scale 1.0, C 16) row; efficiency / ghost rate against the "
                               "generator truth (PAPER.md:199-215); absolute values are not comparable with the "
                               "paper's Table 3 (synthetic events)"},
            "gpu_launches": 2 * steps * len(rows), "sweep": rows}
    print(json.dumps(line), flush=True)


class DeviceWorkload:
    """One synthetic batch resident on the device plus everything the two calls need."""

    def __init__(self, B, geom_tables, batch, params):
        self.B, self.tables, self.batch, self.params = B, geom_tables, batch, params
        self.geom = B.ut_geometry_upload(geom_tables)
        self.hits = B.Hits(batch.hit_capacity, batch.n_events, self.geom)
        self.raw_d, self.bo_d = B.to_device_raw(batch.raw), B.to_device_u32(batch.bank_offsets)
        self.velo = B.VeloStates(batch.velo_x, batch.velo_y, batch.velo_tx, batch.velo_ty, batch.velo_z)
        self.vo_d = B.to_device_u32(batch.velo_offsets)
        self.tracks = B.Tracks(batch.n_velo_total)
        self.config = B.make_config(params)

    def decode(self):
        self.B.ut_decode(self.raw_d, self.bo_d, self.batch.n_events, self.geom, self.hits)

    def compass(self):
        self.B.compass_track(self.hits, self.hits.hit_offsets, self.velo, self.vo_d, self.batch.n_events, self.config,
                             self.tracks)

    def step(self):
        self.decode()
        self.compass()

    def timed(self, torch, flush, steps, warmup):
        """CUDA events on the launch stream around each call of each step, L2 flushed between steps.
        Returns the per-step (decode ms, compass ms, step ms) lists."""
        stream = torch.cuda.current_stream()
        for _ in range(warmup):
            flush.zero_()
            self.step()
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
        torch.cuda.synchronize()
        for k in range(steps):
            flush.zero_()
            ev[k][0].record(stream)
            self.decode()
            ev[k][1].record(stream)
            self.compass()
            ev[k][2].record(stream)
        torch.cuda.synchronize()
        return ([e[0].elapsed_time(e[1]) for e in ev], [e[1].elapsed_time(e[2]) for e in ev],
                [e[0].elapsed_time(e[2]) for e in ev])

    def timed_steps(self, torch, flush, steps, warmup):
        """CUDA events around each step, the two calls back to back (compass_track's programmatic launch behind ut_decode
        needs them adjacent on the stream).  Returns the per-step ms list."""
        stream = torch.cuda.current_stream()
        for _ in range(warmup):
            flush.zero_()
            self.step()
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(steps)]
        torch.cuda.synchronize()
        for k in range(steps):
            flush.zero_()
            ev[k][0].record(stream)
            self.step()
            ev[k][1].record(stream)
        torch.cuda.synchronize()
        return [e[0].elapsed_time(e[1]) for e in ev]

    def facts(self):
        ne, ng = self.batch.n_events, self.tables.n_groups
        n_hits = int(self.hits.hit_offsets[ne * ng].item()) & 0xFFFFFFFF
        status = (int(self.hits.status.item()) | int(self.tracks.status[0].item())) & 0xFFFFFFFF
        return n_hits, status


def two_kernel_ab(B, torch, w, flush, steps):
    """the paper's two-kernel Compass (window ranges as int16 pairs in global memory, then a
    thread-per-track tracklet kernel; Fig. 7) timed beside the fused kernel on the same decoded
    container -- the measurement the paper's own layout claim asks for.  Not part of the step."""
    stream = torch.cuda.current_stream()
    b, T = w.batch, w.batch.n_velo_total
    w.step()
    torch.cuda.synchronize()
    fused_idx = w.tracks.hit_idx[:4 * T].clone()
    out = {}
    for W in (1, 3, 5):
        win = torch.empty(max(T, 1) * 8 * W, dtype=torch.int16, device="cuda")
        st = torch.zeros(1, dtype=torch.int32, device="cuda")
        tr = B.Tracks(T)
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
        for k in range(steps + 2):
            flush.zero_()
            w.decode()                                     # the hits are in L2 as they are for the fused kernel
            e = ev[max(k - 2, 0)]
            e[0].record(stream)
            B.compass_search_windows(w.hits, w.hits.hit_offsets, w.velo, w.vo_d, b.n_events, w.config, W, win, st)
            e[1].record(stream)
            B.compass_tracklets_from_windows(w.hits, w.hits.hit_offsets, w.velo, w.vo_d, b.n_events, w.config, W, win, tr)
            e[2].record(stream)
        torch.cuda.synchronize()
        mw = statistics.mean(e[0].elapsed_time(e[1]) for e in ev)
        mt = statistics.mean(e[1].elapsed_time(e[2]) for e in ev)
        out[f"sectors_{W}"] = {"ms_search_windows": mw, "ms_tracklet_finding": mt, "ms": mw + mt,
                               "tracking_only_events_per_s": b.n_events / (mw + mt) * 1e3,
                               "window_bytes": int(T * 16 * W),
                               "tracklets": int((tr.n_hits[:T] > 0).sum().item()),
                               "equals_fused_kernel": bool(torch.equal(tr.hit_idx[:4 * T], fused_idx))}
    return out


def kernel_table(batch, abytes, md, mc, hbm_peak):
    return {
        "ut_decode_kernel": {"ms": md, "bytes": abytes["decode"], "gbs": abytes["decode"] / md / 1e6,
                             "frac_hbm": abytes["decode"] / md / 1e6 / hbm_peak,
                             "events_per_s": batch.n_events / md * 1e3},
        "compass_kernel": {"ms": mc, "bytes": abytes["compass"], "gbs": abytes["compass"] / mc / 1e6,
                           "frac_hbm": abytes["compass"] / mc / 1e6 / hbm_peak,
                           "events_per_s": batch.n_events / mc * 1e3},
    }


def per_config_report(B, torch, flush, prepared, hbm_peak, steps):
    """north_star: "events/s and achieved fraction of the HBM roofline reported for each [config]".  Device-resident
    inputs, a few steps each; config 5 in its default setting (min_hits 3, scale 1, C 16) on all 10 000 events."""
    rows = {}
    for cid, (cfg, geom_t, batch, params) in prepared.items():
        w = DeviceWorkload(B, geom_t, batch, params)
        t_step = w.timed_steps(torch, flush, steps, 3)                # the step: two calls back to back
        t_dec, t_cmp, _ = w.timed(torch, flush, steps, 0)             # per kernel: an event between the calls
        n_hits, status = w.facts()
        ab = algorithmic_bytes(batch, geom_t, n_hits)
        md, mc, ms = statistics.mean(t_dec), statistics.mean(t_cmp), statistics.mean(t_step)
        k = kernel_table(batch, ab, md, mc, hbm_peak)
        rows[cfg.name] = {
            "events": batch.n_events, "hits": n_hits, "velo_tracks": batch.n_velo_total, "steps": steps,
            "events_per_s": batch.n_events / ms * 1e3, "ms_per_step": ms,
            "decode_only_events_per_s": k["ut_decode_kernel"]["events_per_s"],
            "tracking_only_events_per_s": k["compass_kernel"]["events_per_s"],
            "ms_decode": md, "ms_compass": mc,
            "frac_hbm_decode": k["ut_decode_kernel"]["frac_hbm"], "frac_hbm_compass": k["compass_kernel"]["frac_hbm"],
            "frac_hbm_step": ab["e2e"] / ms / 1e6 / hbm_peak, "gbs_step": ab["e2e"] / ms / 1e6,
            "min_hits": params.min_hits, "max_candidates_per_layer": params.max_candidates_per_layer,
            "status_word": status, "launch": B.last_launch_info()}
        if cid == 4:
            rows[cfg.name]["two_kernel_compass"] = two_kernel_ab(B, torch, w, flush, 3)
        del w
        torch.cuda.empty_cache()
    return rows


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.sweep:
        if rank == 0:
            run_sweep(args, local_rank)
        return

    import synth
    cfg = synth.CONFIGS[args.config]
    n_events = args.events or cfg.n_events
    workers = min(8, os.cpu_count() or 1)
    # generate before CUDA is initialised (the generator may fork workers)
    geom_t, batch, params = synth.make_workload(args.config, n_events=n_events, workers=workers,
                                                first_event=rank * n_events)
    prepared = {}
    if world == 1 and not args.no_per_config and args.events is None:
        for cid in (1, 2, 3, 4, 5):
            if cid != args.config:
                g_, b_, p_ = synth.make_workload(cid, workers=workers)
                prepared[cid] = (synth.CONFIGS[cid], g_, b_, p_)
    import torch
    import torch.distributed as dist
    import __graft_entry__ as entry
    if rank == 0:
        entry.build()
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    torch.cuda.set_device(local_rank)
    from paper_2002_11529_b200 import binding as B
    dev = torch.device("cuda", local_rank)

    w = DeviceWorkload(B, geom_t, batch, params)
    geom, hits, tracks, vo_d, config = w.geom, w.hits, w.tracks, w.vo_d, w.config
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2
    stream = torch.cuda.current_stream()

    w.step()
    torch.cuda.synchronize()
    launches_per_step = 2
    info = B.last_launch_info()
    n_hits, status = w.facts()
    abytes = algorithmic_bytes(batch, geom_t, n_hits)

    if world > 1:
        ne = torch.tensor([batch.n_events], dtype=torch.float64, device=dev)
        dist.all_reduce(ne, op=dist.ReduceOp.SUM)
        events_all = float(ne.item())
    else:
        events_all = float(batch.n_events)

    # (measured before the nvidia-smi clock sampler starts: its polling was seen to slow the host copies)
    # ---- end to end through the host-buffer C-ABI call (H2D + kernels + D2H inside the timed region) ----
    e2e = None
    if not args.no_e2e:
        T = batch.n_velo_total
        # host buffers from the library's own page-locked allocator (ut_host_alloc = cudaHostAlloc): torch's pinned
        # tensors of this size were seen to copy at 12-40 GB/s in some processes on this box, these at 54 GB/s
        pin = B.to_host_pinned
        raw_h = pin(np.concatenate([batch.raw, np.zeros(32, np.uint8)]))
        bo_h, vo_h = pin(batch.bank_offsets.view(np.int32)), pin(batch.velo_offsets.view(np.int32))
        # the four VELO arrays are rows of one allocation, and so are n_hits / qop / chi2: evenly spaced host arrays
        # travel as one strided copy each (the call accepts any four pointers)
        Tp = (max(T, 1) + 63) // 64 * 64
        velo_blk = B.host_tensor(4 * Tp, torch.float32)
        velo_h = [velo_blk[r * Tp:r * Tp + T] for r in range(4)]
        for dst, src in zip(velo_h, (batch.velo_x, batch.velo_y, batch.velo_tx, batch.velo_ty)):
            dst.numpy()[:] = src
        # ... and the track SoA is one [7][T] block (4 rows of hit_idx, n_hits, qop, chi2): one strided copy per chunk
        T1 = max(T, 1)
        res_blk = B.host_tensor(7 * T1, torch.int32)
        out_h = {"hit_idx": res_blk[0:4 * T1], "n_hits": res_blk[4 * T1:5 * T1],
                 "qop": res_blk[5 * T1:6 * T1].view(torch.float32), "chi2": res_blk[6 * T1:7 * T1].view(torch.float32),
                 "status": B.host_tensor(2, torch.int32), "n_hits_total": B.host_tensor(1, torch.int32)}
        out_h["status"].zero_()
        out_h["n_hits_total"].zero_()
        pipe = B.Pipeline(geom, batch.n_events, int(batch.raw.size) + 32, batch.hit_capacity, max(T, 1))
        run = lambda: pipe.run_host(raw_h, int(batch.raw.size), bo_h, velo_h, batch.velo_z, vo_h, T, batch.n_events,
                                    config, out_h)
        for _ in range(3):
            run()
        torch.cuda.synchronize()
        e2e_launches = B.last_launch_info()["kernels_launched"]
        k_e2e = max(10, min(args.steps, 100))
        if world > 1:
            dist.barrier()
        # per step: flush L2 (outside the timed part), then H2D + kernels + D2H + sync through the C ABI
        t_steps = []
        for _ in range(k_e2e):
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            run()
            torch.cuda.synchronize()       # the step's result is on the host before the next one starts
            t_steps.append(time.perf_counter() - t0)
        t_e2e = float(sum(t_steps))
        if world > 1:
            t = torch.tensor([t_e2e], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            t_e2e = float(t.item())
        h2d = int(batch.raw.size) + 4 * (batch.bank_offsets.size + batch.velo_offsets.size) + 16 * T
        e2e = {"value": events_all * k_e2e / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": 28 * T + 12, "steps": k_e2e,
               "ms_per_step_mean": 1e3 * t_e2e / k_e2e, "ms_per_step_median": 1e3 * statistics.median(t_steps),
               "ms_per_step_min": 1e3 * min(t_steps), "kernels_per_step": e2e_launches,
               "api": "ut_pipeline_run_host (pinned host buffers in, host track SoA out, sync per step)"}
        ok = np.array_equal(out_h["n_hits"][:T].numpy(), tracks.n_hits[:T].cpu().numpy())
        e2e["matches_device_path"] = bool(ok)
        e2e["timeline_ms_last_step"] = pipe.timeline()      # device-side events of the last step, per chunk
        pipe.destroy()
        for t_ in [raw_h, bo_h, vo_h, velo_blk, res_blk, out_h["status"], out_h["n_hits_total"]]:
            B.host_free(t_)

    sampler = ClockSampler(local_rank) if rank == 0 and not os.environ.get("BENCH_NO_SAMPLER") else None
    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        w.step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    # The timed region: CUDA events around each step (the two calls back to back, as a user issues them: compass_track is
    # launched with programmatic stream serialization, so its CTAs may take SMs the decode has left and stage their
    # tables while its last events finish -- an event record between the two calls would forbid that).
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    if sampler:
        sampler.mark()
    torch.cuda.synchronize()
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.zero_()
        ev[k][0].record(stream)
        w.decode()
        w.compass()
        ev[k][1].record(stream)
    torch.cuda.synchronize()
    t_wall = time.perf_counter() - t_wall0
    if sampler:
        sampler.mark()
    if world > 1:
        dist.barrier()
    t_step = [e[0].elapsed_time(e[1]) for e in ev]
    # per-kernel times from a second pass with an event between the two calls (no overlap there: decode + Compass of
    # this pass is a few microseconds more than a step of the timed region)
    t_dec, t_cmp, _ = w.timed(torch, flush, min(args.steps, 100), 0)
    total_ms = float(sum(t_step))
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    clocks = sampler.stop() if sampler else None

    # ---- SURVEY.md 8(f) row 1 (not part of the step): compacted track output, timed on its own ----
    compact = B.CompactTracks(batch.n_velo_total, batch.n_velo_total, batch.n_events)
    evc = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(min(args.steps, 50))]
    for _ in range(3):
        B.compass_consolidate(tracks, vo_d, batch.n_events, compact)
    for a_, b_ in evc:
        flush.zero_()
        a_.record(stream)
        B.compass_consolidate(tracks, vo_d, batch.n_events, compact)
        b_.record(stream)
    torch.cuda.synchronize()
    t_cons = statistics.mean(a_.elapsed_time(b_) for a_, b_ in evc)
    n_compact = int(compact.track_offsets[batch.n_events].item())
    ab = two_kernel_ab(B, torch, w, flush, 5) if world == 1 else None
    cons_bytes = 28 * batch.n_velo_total + 4 * (batch.n_events + 1) + 32 * n_compact + 4 * (batch.n_events + 1)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "MEASURED_PEAKS.json hbm_gbs (measured copy)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    md, mc, ms = statistics.mean(t_dec), statistics.mean(t_cmp), statistics.mean(t_step)
    kern = kernel_table(batch, abytes, md, mc, hbm_peak)
    dom = "ut_decode_kernel" if md >= mc else "compass_kernel"
    counters, why_not = (ncu_counters(cfg.name) if batch.n_events == cfg.n_events
                         else (None, "not the workload's full size"))
    roof = {"kernel": dom, "bound": "hbm", "achieved": kern[dom]["gbs"], "peak": hbm_peak, "unit": "GB/s",
            "frac": kern[dom]["frac_hbm"],
            "traffic": counters.get(dom, {}).get("dram_bytes") if counters else None,
            "traffic_source": (f"{counters['source']} (commit {counters['commit']})" if counters else why_not),
            "peak_source": peak_src, "algorithmic_bytes_per_launch": kern[dom]["bytes"], "issue": None,
            "end_to_end": {"bytes": abytes["e2e"], "gbs": abytes["e2e"] / ms / 1e6,
                           "frac": abytes["e2e"] / ms / 1e6 / hbm_peak, "frac_of_8TBs": abytes["e2e"] / ms / 1e6 / 8000.0}}
    if counters:
        issue_peak = 148 * 4 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6          # warp-inst / s
        roof["issue"] = {k: {"warp_inst_per_launch": counters[k]["warp_inst"],
                             "achieved_ginst_s": counters[k]["warp_inst"] / kern[k]["ms"] / 1e6,
                             "peak_ginst_s": issue_peak / 1e9,
                             "frac": counters[k]["warp_inst"] / (kern[k]["ms"] * 1e-3) / issue_peak}
                         for k in kern if k in counters and "warp_inst" in counters[k]}
        roof["issue"]["note"] = ("context: both kernels are issue / latency bound, not HBM bound; instruction counts from "
                                 "the committed ncu capture")
    line = {
        "metric": METRIC, "value": events_all * args.steps / (total_ms * 1e-3), "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "events_per_gpu": batch.n_events, "hits": n_hits,
                   "velo_tracks": batch.n_velo_total, "min_hits": params.min_hits,
                   "max_candidates_per_layer": params.max_candidates_per_layer, "p_min_gev": cfg.p_min_gev,
                   "window_scale": cfg.window_scale, "l2": "flushed (256 MiB memset) between timed steps",
                   "timing": "cuda events around each step (two calls back to back) on the launch stream, sum over steps, max over ranks; per-kernel ms from a second pass with an event between the calls",
                   "status_word": status, "launch": info},
        "clocks": clocks, "gpu_launches": launches_per_step * args.steps, "e2e": e2e,
        "roofline": roof, "kernels": kern,
        "decode_only_events_per_s": kern["ut_decode_kernel"]["events_per_s"],
        "tracking_only_events_per_s": kern["compass_kernel"]["events_per_s"],
        "median_ms": {"decode": statistics.median(t_dec), "compass": statistics.median(t_cmp),
                      "step": statistics.median(t_step), "step_min": min(t_step)},
        "wall_events_per_s_incl_flush": batch.n_events * args.steps / t_wall,
        "next_rows": {"compass_consolidate": {"ms": t_cons, "tracklets": n_compact, "bytes": int(cons_bytes),
                                               "gbs": cons_bytes / t_cons / 1e6,
                                               "frac_hbm": cons_bytes / t_cons / 1e6 / hbm_peak,
                                               "note": "SURVEY.md 8(f) row 1, timed alone, not part of the step"},
                      "two_kernel_compass": {"fused_ms": mc, "variants": ab,
                                             "note": "SURVEY.md 8(f) row 2: the paper's search-windows + thread-per-track "
                                                     "tracklet kernels with int16 window ranges (Fig. 7) on the same "
                                                     "container, timed alone; 5 sector groups = the fused kernel's "
                                                     "results"}},
    }
    if prepared:
        del w
        line["per_config"] = per_config_report(B, torch, flush, prepared, hbm_peak, max(3, min(args.steps, 10)))
        line["per_config"][cfg.name] = "this line (value, kernels, roofline)"
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(batch, geom_t, params)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
