"""ctypes front-end of the CPU oracle (``ut_oracle.cpp``).  TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares nothing with
``paper_2002_11529_b200`` (no code, headers, tables or helpers); both take their
inputs from ``synth``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading
from dataclasses import dataclass

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "ut_oracle.cpp")
_LIB = os.path.join(_DIR, "liboracle.so")
_lib = None
_lock = threading.Lock()

ST_UNKNOWN_SECTOR, ST_DUPLICATE_SECTOR, ST_BAD_BANK_SIZE, ST_CAPACITY = 1, 2, 4, 8


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (no FMA contraction: DESIGN.md A14)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC",
                               "-shared", _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


class _Geometry(C.Structure):
    _fields_ = [("n_layers", C.c_uint32), ("n_sectors", C.c_uint32), ("n_groups", C.c_uint32),
                ("id_table_size", C.c_uint32),
                ("id_to_sector", C.c_void_p), ("sector_raw_id", C.c_void_p), ("sector_group", C.c_void_p),
                ("x0", C.c_void_p), ("pitch", C.c_void_p), ("dxdy", C.c_void_p), ("z", C.c_void_p),
                ("y_begin", C.c_void_p), ("y_end", C.c_void_p), ("weight", C.c_void_p),
                ("group_xmin", C.c_void_p), ("group_xmax", C.c_void_p),
                ("layer_z", C.c_float * 4), ("layer_dxdy", C.c_float * 4),
                ("kick_nx", C.c_uint32), ("kick_ny", C.c_uint32), ("kick_x_lo", C.c_float), ("kick_y_lo", C.c_float),
                ("kick_inv_dx", C.c_float), ("kick_inv_dy", C.c_float), ("kick_z_ref", C.c_float),
                ("kick_kappa", C.c_void_p), ("kick_z_mag", C.c_void_p)]


class _Hits(C.Structure):
    _fields_ = [("x_at_y0", C.c_void_p), ("z_at_y0", C.c_void_p), ("y_begin", C.c_void_p),
                ("y_end", C.c_void_p), ("dxdy", C.c_void_p), ("weight", C.c_void_p), ("id", C.c_void_p),
                ("capacity", C.c_uint64)]


class _Config(C.Structure):
    _fields_ = [("win_half", C.c_float * 4), ("y_tol", C.c_float), ("max_slope", C.c_float),
                ("kink_tol", C.c_float), ("seed_tol", C.c_float), ("w_velo", C.c_float),
                ("max_chi2_ndf", C.c_float), ("kappa", C.c_float), ("z_mag", C.c_float),
                ("min_hits", C.c_int32), ("max_candidates_per_layer", C.c_int32), ("both_directions", C.c_int32)]


def _load():
    global _lib
    with _lock:
        if _lib is None:
            build()
            lib = C.CDLL(_LIB)
            lib.oracle_decode.restype = C.c_int32
            lib.oracle_compass.restype = C.c_int32
            lib.oracle_fit.restype = C.c_int32
            lib.oracle_consolidate.restype = C.c_int32
            lib.oracle_search_windows.restype = C.c_int32
            lib.oracle_compass_from_windows.restype = C.c_int32
            _lib = lib
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _geom_struct(geom):
    keep = [np.ascontiguousarray(getattr(geom, n)) for n in
            ("id_to_sector", "sector_raw_id", "sector_group", "x0", "pitch", "dxdy", "z", "y_begin", "y_end",
             "weight", "group_xmin", "group_xmax")]
    s = _Geometry(geom.n_layers, geom.n_sectors, geom.n_groups, geom.id_table_size, *[_p(a) for a in keep])
    s.layer_z[:] = [float(v) for v in geom.layer_z]
    s.layer_dxdy[:] = [float(v) for v in geom.layer_dxdy]
    lut = getattr(geom, "kick", None)
    if lut is not None:                                   # position-dependent kick table (synth/field.py)
        kk, kz = np.ascontiguousarray(lut.kappa, np.float32), np.ascontiguousarray(lut.z_mag, np.float32)
        keep += [kk, kz]
        s.kick_nx, s.kick_ny = lut.nx, lut.ny
        s.kick_x_lo, s.kick_y_lo, s.kick_inv_dx, s.kick_inv_dy, s.kick_z_ref = lut.x_lo, lut.y_lo, lut.inv_dx, lut.inv_dy, lut.z_ref
        s.kick_kappa, s.kick_z_mag = _p(kk), _p(kz)
    return s, keep


def _config_struct(p):
    c = _Config()
    c.win_half[:] = list(p.win_half)
    for n in ("y_tol", "max_slope", "kink_tol", "seed_tol", "w_velo", "max_chi2_ndf", "kappa", "z_mag",
              "min_hits", "max_candidates_per_layer"):
        setattr(c, n, getattr(p, n))
    c.both_directions = int(getattr(p, "both_directions", 0))
    return c


@dataclass
class Hits:
    x_at_y0: np.ndarray
    z_at_y0: np.ndarray
    y_begin: np.ndarray
    y_end: np.ndarray
    dxdy: np.ndarray
    weight: np.ndarray
    id: np.ndarray
    hit_offsets: np.ndarray      # u32 [n_events*n_groups + 1]
    status: int
    n_hits: int

    FIELDS = ("x_at_y0", "z_at_y0", "y_begin", "y_end", "dxdy", "weight", "id")

    def _struct(self):
        return _Hits(*[_p(getattr(self, f)) for f in self.FIELDS], C.c_uint64(self.x_at_y0.shape[0]))


@dataclass
class Tracks:
    hit_idx: np.ndarray          # i32 [4, T]
    n_hits: np.ndarray           # i32 [T]
    qop: np.ndarray              # f32 [T]
    chi2: np.ndarray             # f32 [T]
    runner_chi2: np.ndarray      # f32 [T]  2nd-best chi2 among valid tracklets with the same n (inf if none)
    cand_n: np.ndarray           # i32 [T, 4] candidates per layer before the cap
    cand_list: np.ndarray        # i32 [T, 4, C] post-cap candidate hit indices (-1 pad)
    n_fits: np.ndarray           # i32 [T]


def decode(raw: np.ndarray, bank_offsets: np.ndarray, n_events: int, geom, capacity: int | None = None,
           order: str = "x") -> Hits:
    """PAPER.md section IV as the plain definition.  order "x": groups sorted by x_at_y0 (A1);
    "y": by (y_begin, x_at_y0) -- the paper's literal Y order."""
    lib = _load()
    raw = np.ascontiguousarray(raw, dtype=np.uint8)
    bank_offsets = np.ascontiguousarray(bank_offsets, dtype=np.uint32)
    if capacity is None:
        capacity = max((int(raw.size) - 6 * n_events * geom.n_sectors) // 2, 0)
    f = lambda: np.zeros(capacity, np.float32)
    h = Hits(f(), f(), f(), f(), f(), f(), np.zeros(capacity, np.uint32),
             np.zeros(n_events * geom.n_groups + 1, np.uint32), 0, 0)
    gs, keep = _geom_struct(geom)
    hs = h._struct()
    st = C.c_uint32(0)
    rc = lib.oracle_decode(_p(raw), _p(bank_offsets), C.c_int32(n_events), C.byref(gs), C.byref(hs),
                           _p(h.hit_offsets), C.byref(st), C.c_int32({"x": 0, "y": 1}[order]))
    if rc != 0:
        raise RuntimeError(f"oracle_decode rc={rc}")
    h.status = int(st.value)
    h.n_hits = int(h.hit_offsets[-1])
    return h


def compass(hits: Hits, velo_x, velo_y, velo_tx, velo_ty, velo_z: float, velo_offsets, n_events: int, geom,
            params, mode: int = 0, event_range: tuple | None = None) -> Tracks:
    """PAPER.md section V step by step.  mode 0 windowed, 1 linear-scan candidates (BF-1),
    2 exhaustive combinations without cap (BF-2)."""
    lib = _load()
    T = int(velo_offsets[n_events])
    Cc = int(params.max_candidates_per_layer)
    out = Tracks(np.full((4, T), -1, np.int32), np.zeros(T, np.int32), np.zeros(T, np.float32),
                 np.zeros(T, np.float32), np.full(T, np.inf, np.float32), np.zeros((T, 4), np.int32),
                 np.full((T, 4, Cc), -1, np.int32), np.zeros(T, np.int32))
    compass_into(out, hits, velo_x, velo_y, velo_tx, velo_ty, velo_z, velo_offsets, n_events, geom, params, mode)
    return out


def compass_into(out: Tracks, hits: Hits, velo_x, velo_y, velo_tx, velo_ty, velo_z, velo_offsets, n_events,
                 geom, params, mode=0, first_event=0, n_sub=None, extras=True):
    """Run events [first_event, first_event+n_sub) writing into ``out`` (disjoint event chunks may run in
    different threads: ctypes releases the GIL)."""
    lib = _load()
    n_sub = n_events - first_event if n_sub is None else n_sub
    velo_offsets = np.ascontiguousarray(velo_offsets, dtype=np.uint32)
    gs, keep = _geom_struct(geom)
    cs = _config_struct(params)
    hs = hits._struct()
    vo = velo_offsets[first_event:]
    ho = hits.hit_offsets[first_event * geom.n_groups:]
    T = out.n_hits.shape[0]
    # outputs are indexed by global track id; hit_idx rows have stride T, so pass the base pointers
    rc = lib.oracle_compass(
        C.c_int32(mode), C.byref(hs), _p(ho), _p(np.ascontiguousarray(velo_x, np.float32)),
        _p(np.ascontiguousarray(velo_y, np.float32)), _p(np.ascontiguousarray(velo_tx, np.float32)),
        _p(np.ascontiguousarray(velo_ty, np.float32)), C.c_float(velo_z), _p(vo), C.c_int32(n_sub),
        C.byref(gs), C.byref(cs), _p(out.hit_idx), _p(out.n_hits), _p(out.qop), _p(out.chi2),
        _p(out.runner_chi2) if extras else None, _p(out.cand_n) if extras else None,
        _p(out.cand_list) if extras and mode != 2 else None, _p(out.n_fits) if extras else None,
        C.c_int64(T))
    if rc != 0:
        raise RuntimeError(f"oracle_compass rc={rc}")


def fit(d, z, w, params):
    """Step 6 alone: returns (a, b, chi2, qop) as float32 scalars."""
    lib = _load()
    d, z, w = (np.ascontiguousarray(v, np.float32) for v in (d, z, w))
    cs = _config_struct(params)
    a, b, c2, q = C.c_float(), C.c_float(), C.c_float(), C.c_float()
    rc = lib.oracle_fit(C.c_int32(len(d)), _p(d), _p(z), _p(w), C.byref(cs), C.byref(a), C.byref(b),
                        C.byref(c2), C.byref(q))
    if rc != 0:
        raise RuntimeError(f"oracle_fit rc={rc}")
    return np.float32(a.value), np.float32(b.value), np.float32(c2.value), np.float32(q.value)


def run_batch(batch, geom, params, mode: int = 0):
    """Decode + Compass on a synth.Batch; returns (Hits, Tracks)."""
    h = decode(batch.raw, batch.bank_offsets, batch.n_events, geom, batch.hit_capacity)
    t = compass(h, batch.velo_x, batch.velo_y, batch.velo_tx, batch.velo_ty, batch.velo_z, batch.velo_offsets,
                batch.n_events, geom, params, mode)
    return h, t


@dataclass
class CompactTracks:
    velo_index: np.ndarray       # u32 [K]
    hit_idx: np.ndarray          # i32 [4, K]
    n_hits: np.ndarray           # i32 [K]
    qop: np.ndarray              # f32 [K]
    chi2: np.ndarray             # f32 [K]
    track_offsets: np.ndarray    # u32 [n_events + 1]
    status: int


def consolidate(hit_idx, n_hits, qop, chi2, velo_offsets, n_events: int, capacity: int | None = None) -> CompactTracks:
    """PAPER.md:460 as the plain definition: keep the tracks with a tracklet, in order."""
    lib = _load()
    T = int(velo_offsets[n_events])
    cap = T if capacity is None else int(capacity)
    hit_idx = np.ascontiguousarray(hit_idx, np.int32).reshape(4, T)
    n_hits, qop, chi2 = (np.ascontiguousarray(n_hits, np.int32), np.ascontiguousarray(qop, np.float32),
                         np.ascontiguousarray(chi2, np.float32))
    vo = np.ascontiguousarray(velo_offsets, np.uint32)
    o_v = np.zeros(max(cap, 1), np.uint32); o_i = np.full((4, max(cap, 1)), -1, np.int32)
    o_n = np.zeros(max(cap, 1), np.int32); o_q = np.zeros(max(cap, 1), np.float32); o_c = np.zeros(max(cap, 1), np.float32)
    off = np.zeros(n_events + 1, np.uint32)
    st = C.c_uint32(0)
    rc = lib.oracle_consolidate(_p(hit_idx), _p(n_hits), _p(qop), _p(chi2), _p(vo), C.c_int32(n_events), _p(o_v),
                                _p(o_i), _p(o_n), _p(o_q), _p(o_c), C.c_uint64(cap), _p(off), C.byref(st))
    if rc != 0:
        raise RuntimeError(f"oracle_consolidate rc={rc}")
    K = min(int(off[-1]), cap)
    return CompactTracks(o_v[:K], o_i[:, :K] if cap else o_i[:, :0], o_n[:K], o_q[:K], o_c[:K], off, int(st.value))


def search_windows(hits: Hits, velo_x, velo_y, velo_tx, velo_ty, velo_z: float, velo_offsets, n_events: int, geom,
                   params, n_sectors_search: int):
    """PAPER.md:286-322 as the plain definition: window ranges as signed 16-bit (begin, size)
    per track x panel x {1, 3, 5} sector groups in the layout of Fig. 7: i16 [T, 4, 2W] (W begins, then W sizes;
    begin relative to the event's first hit; (-1, -1) = no hits).  Returns (windows, status)."""
    lib = _load()
    W = int(n_sectors_search)
    velo_offsets = np.ascontiguousarray(velo_offsets, dtype=np.uint32)
    T = int(velo_offsets[n_events])
    win = np.full((max(T, 1), 4, 2 * W), -9, np.int16)
    gs, keep = _geom_struct(geom)
    cs = _config_struct(params)
    hs = hits._struct()
    st = C.c_uint32(0)
    f = lambda a: _p(np.ascontiguousarray(a, np.float32))
    rc = lib.oracle_search_windows(C.byref(hs), _p(hits.hit_offsets), f(velo_x), f(velo_y), f(velo_tx), f(velo_ty),
                                   C.c_float(velo_z), _p(velo_offsets), C.c_int32(n_events), C.byref(gs), C.byref(cs),
                                   C.c_int32(W), _p(win), C.byref(st))
    if rc != 0:
        raise RuntimeError(f"oracle_search_windows rc={rc}")
    return win[:T], int(st.value)


def compass_from_windows(hits: Hits, windows, velo_x, velo_y, velo_tx, velo_ty, velo_z: float, velo_offsets,
                         n_events: int, geom, params, n_sectors_search: int) -> Tracks:
    """PAPER.md:324-348 from stored window ranges.  cand_n = candidates per layer before the cap."""
    lib = _load()
    W = int(n_sectors_search)
    velo_offsets = np.ascontiguousarray(velo_offsets, dtype=np.uint32)
    T = int(velo_offsets[n_events])
    out = Tracks(np.full((4, T), -1, np.int32), np.zeros(T, np.int32), np.zeros(T, np.float32), np.zeros(T, np.float32),
                 None, np.zeros((T, 4), np.int32), None, None)
    gs, keep = _geom_struct(geom)
    cs = _config_struct(params)
    hs = hits._struct()
    win = np.ascontiguousarray(windows, np.int16)
    f = lambda a: _p(np.ascontiguousarray(a, np.float32))
    rc = lib.oracle_compass_from_windows(C.byref(hs), _p(hits.hit_offsets), f(velo_x), f(velo_y), f(velo_tx), f(velo_ty),
                                         C.c_float(velo_z), _p(velo_offsets), C.c_int32(n_events), C.byref(gs),
                                         C.byref(cs), C.c_int32(W), _p(win), _p(out.hit_idx), _p(out.n_hits), _p(out.qop),
                                         _p(out.chi2), _p(out.cand_n))
    if rc != 0:
        raise RuntimeError(f"oracle_compass_from_windows rc={rc}")
    return out
