"""ctypes binding of libutcompass.so with the same names as include/ut_compass.h.

PyTorch is used for device memory and streams only.  Nothing here computes: each function
marshals pointers and calls the C ABI.  Missing library => ImportError (no fallback).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

from . import build as _build

_LIBPATH = _build.LIB
if not os.path.exists(_LIBPATH):
    raise ImportError(f"{_LIBPATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                      "(nvcc, sm_100a). There is no CPU fallback.")
_lib = C.CDLL(_LIBPATH)

UT_OK = 0
UT_ERR_NULL, UT_ERR_ARG, UT_ERR_GEOMETRY, UT_ERR_CUDA, UT_ERR_LIMIT = -1, -2, -3, -4, -5
UT_STATUS_UNKNOWN_SECTOR, UT_STATUS_DUPLICATE_SECTOR, UT_STATUS_BAD_BANK_SIZE, UT_STATUS_CAPACITY = 1, 2, 4, 8
UT_STATUS_BAD_OFFSETS, UT_STATUS_EVENT_TOO_LARGE, UT_STATUS_BAD_HIT_ID = 16, 32, 64
UT_MAX_CANDIDATES = 32
UT_ORDER_X, UT_ORDER_Y = 0, 1


class ut_geometry(C.Structure):
    _fields_ = [("n_layers", C.c_uint32), ("n_sectors", C.c_uint32), ("n_groups", C.c_uint32),
                ("id_table_size", C.c_uint32),
                ("id_to_sector", C.c_void_p), ("sector_raw_id", C.c_void_p), ("sector_group", C.c_void_p),
                ("x0", C.c_void_p), ("pitch", C.c_void_p), ("dxdy", C.c_void_p), ("z", C.c_void_p),
                ("y_begin", C.c_void_p), ("y_end", C.c_void_p), ("weight", C.c_void_p),
                ("group_xmin", C.c_void_p), ("group_xmax", C.c_void_p),
                ("layer_z", C.c_float * 4), ("layer_dxdy", C.c_float * 4),
                ("group_first_sector", C.c_void_p), ("sector_rows", C.c_void_p), ("sector_yorder", C.c_void_p),
                ("flags", C.c_uint32),
                ("owner", C.c_void_p),
                ("kick_nx", C.c_uint32), ("kick_ny", C.c_uint32), ("kick_x_lo", C.c_float), ("kick_y_lo", C.c_float),
                ("kick_inv_dx", C.c_float), ("kick_inv_dy", C.c_float), ("kick_z_ref", C.c_float),
                ("kick_kappa", C.c_void_p), ("kick_z_mag", C.c_void_p), ("layer_weight", C.c_float * 4)]


class ut_hits(C.Structure):
    _fields_ = [("x_at_y0", C.c_void_p), ("z_at_y0", C.c_void_p), ("y_begin", C.c_void_p), ("y_end", C.c_void_p),
                ("dxdy", C.c_void_p), ("weight", C.c_void_p), ("id", C.c_void_p), ("capacity", C.c_uint64),
                ("geom", C.POINTER(ut_geometry)), ("status", C.c_void_p), ("workspace", C.c_void_p),
                ("x_by_sector", C.c_void_p), ("idx_by_sector", C.c_void_p), ("sector_offsets", C.c_void_p),
                ("order", C.c_uint32)]


class velo_states(C.Structure):
    _fields_ = [("x", C.c_void_p), ("y", C.c_void_p), ("tx", C.c_void_p), ("ty", C.c_void_p), ("z", C.c_float)]


class compass_config(C.Structure):
    _fields_ = [("win_half", C.c_float * 4), ("y_tol", C.c_float), ("max_slope", C.c_float),
                ("kink_tol", C.c_float), ("seed_tol", C.c_float), ("w_velo", C.c_float),
                ("max_chi2_ndf", C.c_float), ("kappa", C.c_float), ("z_mag", C.c_float),
                ("min_hits", C.c_int32), ("max_candidates_per_layer", C.c_int32), ("both_directions", C.c_int32)]


class ut_tracks(C.Structure):
    _fields_ = [("hit_idx", C.c_void_p), ("n_hits", C.c_void_p), ("qop", C.c_void_p), ("chi2", C.c_void_p),
                ("status", C.c_void_p)]


class ut_compact_tracks(C.Structure):
    _fields_ = [("velo_index", C.c_void_p), ("hit_idx", C.c_void_p), ("n_hits", C.c_void_p), ("qop", C.c_void_p),
                ("chi2", C.c_void_p), ("capacity", C.c_uint64), ("status", C.c_void_p), ("workspace", C.c_void_p),
                ("max_velo_total", C.c_uint32)]


class ut_tuning(C.Structure):
    _fields_ = [(n, C.c_int32) for n in
                ("decode_block", "decode_raw_stage_bytes", "decode_sort_buf", "decode_max_ctas_per_sm", "compass_block",
                 "compass_hit_stage", "compass_trk_stage", "compass_split", "pipeline_chunk_events",
                 "compass_interval_min", "pipeline_zero_copy", "decode_hit_stage", "compass_event_order")] + \
               [("reserved", C.c_int32 * 3)]


class ut_launch_info(C.Structure):
    _fields_ = [(n, C.c_int32) for n in
                ("kernels_launched", "decode_grid", "decode_block", "decode_smem_bytes", "decode_raw_stage_bytes",
                 "decode_sort_buf", "compass_grid", "compass_block", "compass_smem_bytes", "compass_hit_stage",
                 "compass_split", "compass_view", "decode_hit_stage", "compass_event_order")]


EXPORTS = ["ut_version", "ut_last_error", "ut_last_launch_info", "ut_tuning_get", "ut_tuning_set",
           "ut_sector_offsets_stride", "compass_search_windows", "compass_tracklets_from_windows", "ut_geometry_upload", "ut_geometry_free",
           "ut_decode_workspace_bytes", "ut_decode_workspace_init", "ut_decode", "compass_config_default",
           "compass_track", "compass_consolidate", "compass_consolidate_workspace_bytes", "ut_pipeline_create", "ut_pipeline_destroy", "ut_pipeline_run_host",
           "ut_pipeline_device_hits", "ut_host_alloc", "ut_host_free", "ut_pipeline_timeline", "ut_decode_static"]

_lib.ut_version.restype = C.c_char_p
_lib.ut_last_error.restype = C.c_char_p
_lib.ut_decode_workspace_bytes.restype = C.c_size_t
_lib.ut_decode_workspace_bytes.argtypes = [C.c_int32, C.c_void_p]
_lib.ut_decode_workspace_init.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
_lib.ut_geometry_upload.argtypes = [C.POINTER(ut_geometry), C.POINTER(ut_geometry)]
_lib.ut_geometry_free.argtypes = [C.POINTER(ut_geometry)]
_lib.ut_decode.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(ut_geometry), C.POINTER(ut_hits),
                           C.c_void_p, C.c_void_p]
_lib.ut_decode_static.argtypes = _lib.ut_decode.argtypes
_lib.compass_config_default.argtypes = [C.c_float, C.c_float, C.c_int32, C.c_int32, C.POINTER(ut_geometry),
                                        C.POINTER(compass_config)]
_lib.compass_track.argtypes = [C.POINTER(ut_hits), C.c_void_p, C.POINTER(velo_states), C.c_void_p, C.c_int32,
                               C.POINTER(compass_config), C.POINTER(ut_tracks), C.c_void_p]
_lib.compass_search_windows.argtypes = [C.POINTER(ut_hits), C.c_void_p, C.POINTER(velo_states), C.c_void_p, C.c_int32,
                                        C.POINTER(compass_config), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.compass_tracklets_from_windows.argtypes = [C.POINTER(ut_hits), C.c_void_p, C.POINTER(velo_states), C.c_void_p,
                                                C.c_int32, C.POINTER(compass_config), C.c_int32, C.c_void_p,
                                                C.POINTER(ut_tracks), C.c_void_p]
_lib.compass_consolidate_workspace_bytes.restype = C.c_size_t
_lib.compass_consolidate_workspace_bytes.argtypes = [C.c_uint32]
_lib.compass_consolidate.argtypes = [C.POINTER(ut_tracks), C.c_void_p, C.c_int32, C.POINTER(ut_compact_tracks),
                                     C.c_void_p, C.c_void_p]
_lib.ut_pipeline_create.argtypes = [C.POINTER(ut_geometry), C.c_int32, C.c_size_t, C.c_uint64, C.c_uint32,
                                    C.POINTER(C.c_void_p)]
_lib.ut_pipeline_destroy.argtypes = [C.c_void_p]
_lib.ut_pipeline_run_host.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(velo_states),
                                      C.c_void_p, C.c_uint32, C.c_int32, C.POINTER(compass_config),
                                      C.POINTER(ut_tracks), C.c_void_p, C.c_void_p, C.c_void_p]
_lib.ut_pipeline_device_hits.argtypes = [C.c_void_p, C.POINTER(ut_hits), C.POINTER(C.c_void_p)]
_lib.ut_pipeline_timeline.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.POINTER(C.c_int32)]
_lib.ut_host_alloc.argtypes = [C.POINTER(C.c_void_p), C.c_size_t]
_lib.ut_host_free.argtypes = [C.c_void_p]
_lib.ut_last_launch_info.argtypes = [C.POINTER(ut_launch_info)]
_lib.ut_sector_offsets_stride.restype = C.c_uint32
_lib.ut_sector_offsets_stride.argtypes = [C.POINTER(ut_geometry)]
_lib.ut_tuning_get.argtypes = [C.POINTER(ut_tuning)]
_lib.ut_tuning_set.argtypes = [C.POINTER(ut_tuning)]
for _n in EXPORTS:
    if _n not in ("ut_version", "ut_last_error", "ut_decode_workspace_bytes", "ut_last_launch_info",
                  "compass_consolidate_workspace_bytes", "ut_sector_offsets_stride"):
        getattr(_lib, _n).restype = C.c_int32


class UTError(RuntimeError):
    pass


def _check(rc, what):
    if rc != UT_OK:
        raise UTError(f"{what} failed with code {rc} {_lib.ut_last_error().decode()}")


def ut_version() -> str:
    return _lib.ut_version().decode()


def _stream_ptr(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


_GEOM_ARRAYS = (("id_to_sector", np.uint32), ("sector_raw_id", np.uint32), ("sector_group", np.uint32),
                ("x0", np.float32), ("pitch", np.float32), ("dxdy", np.float32), ("z", np.float32),
                ("y_begin", np.float32), ("y_end", np.float32), ("weight", np.float32),
                ("group_xmin", np.float32), ("group_xmax", np.float32))


class Geometry:
    """Device-resident geometry tables (ut_geometry_upload / ut_geometry_free)."""

    def __init__(self, tables):
        host = ut_geometry()
        keep = []
        host.n_layers, host.n_sectors, host.n_groups = tables.n_layers, tables.n_sectors, tables.n_groups
        host.id_table_size = int(np.asarray(tables.id_to_sector).shape[0])
        for name, dt in _GEOM_ARRAYS:
            arr = np.ascontiguousarray(getattr(tables, name), dtype=dt)
            keep.append(arr)
            setattr(host, name, arr.ctypes.data)
        host.layer_z[:] = [float(v) for v in tables.layer_z]
        host.layer_dxdy[:] = [float(v) for v in tables.layer_dxdy]
        lut = getattr(tables, "kick", None)
        if lut is not None:                                # optional position-dependent kick table
            kk, kz = np.ascontiguousarray(lut.kappa, np.float32), np.ascontiguousarray(lut.z_mag, np.float32)
            keep += [kk, kz]
            host.kick_nx, host.kick_ny = lut.nx, lut.ny
            host.kick_x_lo, host.kick_y_lo, host.kick_inv_dx, host.kick_inv_dy = lut.x_lo, lut.y_lo, lut.inv_dx, lut.inv_dy
            host.kick_z_ref = lut.z_ref
            host.kick_kappa, host.kick_z_mag = kk.ctypes.data, kz.ctypes.data
        self.c = ut_geometry()
        _check(_lib.ut_geometry_upload(C.byref(host), C.byref(self.c)), "ut_geometry_upload")
        self.n_sectors, self.n_groups = tables.n_sectors, tables.n_groups

    def free(self):
        if self.c.owner:
            _lib.ut_geometry_free(C.byref(self.c))

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def ut_geometry_upload(tables) -> Geometry:
    return Geometry(tables)


def ut_sector_offsets_stride(geometry: "Geometry") -> int:
    return int(_lib.ut_sector_offsets_stride(C.byref(geometry.c)))


def ut_decode_workspace_bytes(max_events: int, geometry: "Geometry | None" = None) -> int:
    return int(_lib.ut_decode_workspace_bytes(max_events, C.byref(geometry.c) if geometry is not None else None))


class Hits:
    """Caller-owned SoA hit container on the device (torch tensors) + its ut_hits descriptor."""
    FIELDS = ("x_at_y0", "z_at_y0", "y_begin", "y_end", "dxdy", "weight", "id")

    def __init__(self, capacity: int, max_events: int, geometry: Geometry, device="cuda", sector_view: bool = True,
                 order: str = "x"):
        """sector_view: also allocate the optional per-sector view (x_by_sector, idx_by_sector, sector_offsets)
        that ut_decode fills for compass_track."""
        self.capacity = int(capacity)
        self.order = {"x": UT_ORDER_X, "y": UT_ORDER_Y}[order]
        n = max(self.capacity, 1)
        self.x_at_y0, self.z_at_y0, self.y_begin, self.y_end, self.dxdy, self.weight = (
            torch.empty(n, dtype=torch.float32, device=device) for _ in range(6))
        self.id = torch.empty(n, dtype=torch.int32, device=device)
        self.status = torch.zeros(1, dtype=torch.int32, device=device)
        nbytes = ut_decode_workspace_bytes(max_events, geometry)
        self.workspace = torch.zeros((nbytes + 15) // 16 * 2, dtype=torch.int64, device=device)   # zeroed once
        self.hit_offsets = torch.zeros(max_events * geometry.n_groups + 1, dtype=torch.int32, device=device)
        self.geometry = geometry
        self.x_by_sector = self.idx_by_sector = self.sector_offsets = None
        if sector_view:
            n8 = (n + 7) // 8 * 8
            self.x_by_sector = torch.empty(n8, dtype=torch.float32, device=device)
            self.idx_by_sector = torch.empty(n8, dtype=torch.int16, device=device)
            self.sector_offsets = torch.zeros(max(max_events, 1) * ut_sector_offsets_stride(geometry), dtype=torch.int16,
                                              device=device)
        self.c = self.descriptor()

    def descriptor(self) -> "ut_hits":
        ptr = lambda t: t.data_ptr() if t is not None else None
        return ut_hits(self.x_at_y0.data_ptr(), self.z_at_y0.data_ptr(), self.y_begin.data_ptr(),
                       self.y_end.data_ptr(), self.dxdy.data_ptr(), self.weight.data_ptr(), self.id.data_ptr(),
                       self.capacity, C.pointer(self.geometry.c), self.status.data_ptr(), self.workspace.data_ptr(),
                       ptr(self.x_by_sector), ptr(self.idx_by_sector), ptr(self.sector_offsets), self.order)


class Tracks:
    def __init__(self, n_velo_total: int, device="cuda"):
        n = max(int(n_velo_total), 1)
        self.n = int(n_velo_total)
        self.hit_idx = torch.empty(4 * n, dtype=torch.int32, device=device)
        self.n_hits = torch.empty(n, dtype=torch.int32, device=device)
        self.qop = torch.empty(n, dtype=torch.float32, device=device)
        self.chi2 = torch.empty(n, dtype=torch.float32, device=device)
        self.status = torch.zeros(4, dtype=torch.int32, device=device)     # [0] status word, [1..3] kernel scratch
        self.c = ut_tracks(self.hit_idx.data_ptr(), self.n_hits.data_ptr(), self.qop.data_ptr(),
                           self.chi2.data_ptr(), self.status.data_ptr())

    def numpy(self):
        n = self.n
        return (self.hit_idx[:4 * n].cpu().numpy().reshape(4, n), self.n_hits[:n].cpu().numpy(),
                self.qop[:n].cpu().numpy(), self.chi2[:n].cpu().numpy())


class CompactTracks:
    """Caller-owned compacted track container (compass_consolidate) + the per-event offsets."""

    def __init__(self, capacity: int, max_velo_total: int, max_events: int, device="cuda"):
        n = max(int(capacity), 1)
        self.capacity = int(capacity)
        self.velo_index = torch.empty(n, dtype=torch.int32, device=device)
        self.hit_idx = torch.empty(4 * n, dtype=torch.int32, device=device)
        self.n_hits = torch.empty(n, dtype=torch.int32, device=device)
        self.qop = torch.empty(n, dtype=torch.float32, device=device)
        self.chi2 = torch.empty(n, dtype=torch.float32, device=device)
        self.status = torch.zeros(1, dtype=torch.int32, device=device)
        nbytes = int(_lib.compass_consolidate_workspace_bytes(int(max_velo_total)))
        self.workspace = torch.zeros((nbytes + 15) // 16 * 2, dtype=torch.int64, device=device)   # zeroed once
        self.track_offsets = torch.zeros(max_events + 1, dtype=torch.int32, device=device)
        self.c = ut_compact_tracks(self.velo_index.data_ptr(), self.hit_idx.data_ptr(), self.n_hits.data_ptr(),
                                   self.qop.data_ptr(), self.chi2.data_ptr(), self.capacity, self.status.data_ptr(),
                                   self.workspace.data_ptr(), int(max_velo_total))

    def numpy(self, n_events: int):
        off = self.track_offsets[:n_events + 1].cpu().numpy().view(np.uint32)
        k = min(int(off[-1]), self.capacity)
        cap = max(self.capacity, 1)
        return dict(velo_index=self.velo_index[:k].cpu().numpy().view(np.uint32),
                    hit_idx=self.hit_idx.cpu().numpy().reshape(4, cap)[:, :k], n_hits=self.n_hits[:k].cpu().numpy(),
                    qop=self.qop[:k].cpu().numpy(), chi2=self.chi2[:k].cpu().numpy(), track_offsets=off,
                    status=int(self.status.item()) & 0xFFFFFFFF)


def compass_consolidate(tracks: Tracks, velo_offsets: torch.Tensor, n_events: int, out: CompactTracks,
                        stream=None) -> int:
    rc = _lib.compass_consolidate(C.byref(tracks.c), velo_offsets.data_ptr(), n_events, C.byref(out.c),
                                  out.track_offsets.data_ptr(), _stream_ptr(stream))
    _check(rc, "compass_consolidate")
    return rc


def compass_consolidate_workspace_bytes(max_velo_total: int) -> int:
    return int(_lib.compass_consolidate_workspace_bytes(int(max_velo_total)))


def make_config(params) -> compass_config:
    """compass_config from any object with the fields of include/ut_compass.h (e.g. synth.CompassParams)."""
    c = compass_config()
    c.win_half[:] = list(params.win_half)
    for n in ("y_tol", "max_slope", "kink_tol", "seed_tol", "w_velo", "max_chi2_ndf", "kappa", "z_mag",
              "min_hits", "max_candidates_per_layer"):
        setattr(c, n, getattr(params, n))
    c.both_directions = int(getattr(params, "both_directions", 0))
    return c


def compass_config_default(p_min_mev: float, window_scale: float, min_hits: int, max_candidates_per_layer: int,
                           geometry: Geometry) -> compass_config:
    c = compass_config()
    _check(_lib.compass_config_default(p_min_mev, window_scale, min_hits, max_candidates_per_layer,
                                       C.byref(geometry.c), C.byref(c)), "compass_config_default")
    return c


def ut_decode(raw_banks: torch.Tensor, bank_offsets: torch.Tensor, n_events: int, geometry: Geometry,
              hits_out: Hits, hit_offsets_out: torch.Tensor | None = None, stream=None) -> int:
    """raw_banks: u8 device tensor (16-byte padded); bank_offsets: i32/u32 device tensor."""
    ho = hits_out.hit_offsets if hit_offsets_out is None else hit_offsets_out
    rc = _lib.ut_decode(raw_banks.data_ptr(), bank_offsets.data_ptr(), n_events, C.byref(geometry.c),
                        C.byref(hits_out.c), ho.data_ptr(), _stream_ptr(stream))
    _check(rc, "ut_decode")
    return rc


UT_DECODE_STATIC_MAX_EVENTS = 16384


def ut_decode_static(raw_banks: torch.Tensor, bank_offsets: torch.Tensor, n_events: int, geometry: Geometry,
                     hits_out: Hits, hit_offsets_out: torch.Tensor | None = None, stream=None) -> int:
    """ut_decode with the kernel's scratch in the library's built-in device array (include/ut_compass.h): no device
    allocation anywhere in the call, at most UT_DECODE_STATIC_MAX_EVENTS events, calls on one GPU must not overlap.
    The container's own workspace is not handed over (the descriptor goes in with workspace = NULL)."""
    ho = hits_out.hit_offsets if hit_offsets_out is None else hit_offsets_out
    d = hits_out.descriptor()
    d.workspace = None
    rc = _lib.ut_decode_static(raw_banks.data_ptr(), bank_offsets.data_ptr(), n_events, C.byref(geometry.c),
                               C.byref(d), ho.data_ptr(), _stream_ptr(stream))
    _check(rc, "ut_decode_static")
    return rc


def compass_track(hits: Hits, hit_offsets: torch.Tensor, velo: "VeloStates", velo_offsets: torch.Tensor,
                  n_events: int, config: compass_config, tracks_out: Tracks, stream=None) -> int:
    rc = _lib.compass_track(C.byref(hits.c), hit_offsets.data_ptr(), C.byref(velo.c), velo_offsets.data_ptr(),
                            n_events, C.byref(config), C.byref(tracks_out.c), _stream_ptr(stream))
    _check(rc, "compass_track")
    return rc


def compass_search_windows(hits: Hits, hit_offsets: torch.Tensor, velo: "VeloStates", velo_offsets: torch.Tensor,
                           n_events: int, config: compass_config, n_sectors_search: int, windows_out: torch.Tensor,
                           status: torch.Tensor, stream=None) -> int:
    """windows_out: int16 device tensor [n_velo_total * 4 * 2 * n_sectors_search] (Fig. 7 layout); status: int32[1]."""
    rc = _lib.compass_search_windows(C.byref(hits.c), hit_offsets.data_ptr(), C.byref(velo.c), velo_offsets.data_ptr(),
                                     n_events, C.byref(config), n_sectors_search, windows_out.data_ptr(),
                                     status.data_ptr(), _stream_ptr(stream))
    _check(rc, "compass_search_windows")
    return rc


def compass_tracklets_from_windows(hits: Hits, hit_offsets: torch.Tensor, velo: "VeloStates", velo_offsets: torch.Tensor,
                                   n_events: int, config: compass_config, n_sectors_search: int, windows: torch.Tensor,
                                   tracks_out: Tracks, stream=None) -> int:
    rc = _lib.compass_tracklets_from_windows(C.byref(hits.c), hit_offsets.data_ptr(), C.byref(velo.c),
                                             velo_offsets.data_ptr(), n_events, C.byref(config), n_sectors_search,
                                             windows.data_ptr(), C.byref(tracks_out.c), _stream_ptr(stream))
    _check(rc, "compass_tracklets_from_windows")
    return rc


class VeloStates:
    def __init__(self, x, y, tx, ty, z: float, device="cuda"):
        t = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float32)).to(device) if not isinstance(a, torch.Tensor) else a
        self.x, self.y, self.tx, self.ty = t(x), t(y), t(tx), t(ty)
        if self.x.numel() == 0:
            self.x = self.y = self.tx = self.ty = torch.zeros(1, dtype=torch.float32, device=device)
        self.c = velo_states(self.x.data_ptr(), self.y.data_ptr(), self.tx.data_ptr(), self.ty.data_ptr(), float(z))


def to_device_raw(raw: np.ndarray, device="cuda") -> torch.Tensor:
    """u8 tensor padded to a multiple of 16 bytes (the ABI's read-ahead contract)."""
    n = int(raw.size)
    t = torch.zeros((n + 15) // 16 * 16 + 16, dtype=torch.uint8, device=device)
    if n:
        t[:n] = torch.from_numpy(np.ascontiguousarray(raw))
    return t


def to_device_u32(a: np.ndarray, device="cuda") -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint32).view(np.int32)).to(device)


def ut_tuning_get() -> ut_tuning:
    t = ut_tuning()
    _check(_lib.ut_tuning_get(C.byref(t)), "ut_tuning_get")
    return t


def ut_tuning_set(tuning: "ut_tuning | None" = None, **fields) -> None:
    """Replace the process-wide launch tuning (None and no fields: back to the environment's values; fields given
    by name override the current values).  Results never depend on it."""
    if tuning is None and fields:
        tuning = ut_tuning_get()
    if tuning is not None:
        for k, v in fields.items():
            setattr(tuning, k, int(v))
    _check(_lib.ut_tuning_set(C.byref(tuning) if tuning is not None else None), "ut_tuning_set")


def last_launch_info() -> dict:
    li = ut_launch_info()
    _lib.ut_last_launch_info(C.byref(li))
    return {n: getattr(li, n) for n, _ in ut_launch_info._fields_}


class _HostBlock:
    """One ut_host_alloc allocation; freed when the last tensor that views it is gone."""

    def __init__(self, nbytes: int):
        self.p = C.c_void_p()
        _check(_lib.ut_host_alloc(C.byref(self.p), max(int(nbytes), 1)), "ut_host_alloc")
        self.buf = (C.c_uint8 * max(int(nbytes), 1)).from_address(self.p.value)

    def __del__(self):
        try:
            if self.p:
                _lib.ut_host_free(self.p)
                self.p = C.c_void_p()
        except Exception:
            pass


def host_tensor(n: int, dtype: torch.dtype) -> torch.Tensor:
    """A HOST tensor of n elements in ut_host_alloc memory (page-locked), for ut_pipeline_run_host."""
    blk = _HostBlock(n * torch.empty(0, dtype=dtype).element_size())
    arr = np.frombuffer(blk.buf, dtype=np.uint8)
    t = torch.from_numpy(arr).view(dtype)[:n] if n > 0 else torch.empty(0, dtype=dtype)
    _host_blocks[t.data_ptr()] = blk            # the block lives as long as the process keeps the key; see host_free
    return t


def host_free(t: torch.Tensor) -> None:
    _host_blocks.pop(t.data_ptr(), None)


_host_blocks: dict = {}


def to_host_pinned(a) -> torch.Tensor:
    """Copy of a numpy array in ut_host_alloc memory."""
    a = np.ascontiguousarray(a)
    t = host_tensor(a.size, torch.from_numpy(a[:0].copy()).dtype if a.size == 0 else torch.from_numpy(a.ravel()[:1].copy()).dtype)
    if a.size:
        t.numpy()[:] = a.ravel()
    return t


class Pipeline:
    """ut_pipeline_*: host buffers in, host track SoA out (copies inside the call)."""

    def __init__(self, geometry: Geometry, max_events: int, max_raw_bytes: int, max_hits: int, max_velo: int):
        self.h = C.c_void_p()
        self.geometry = geometry
        _check(_lib.ut_pipeline_create(C.byref(geometry.c), max_events, max_raw_bytes, max_hits, max_velo,
                                       C.byref(self.h)), "ut_pipeline_create")

    def run_host(self, raw_h: torch.Tensor, raw_bytes: int, bank_offsets_h: torch.Tensor, velo_h, velo_z: float,
                 velo_offsets_h: torch.Tensor, n_velo: int, n_events: int, config: compass_config, out_h: dict,
                 stream=None):
        """All tensors are (pinned) HOST tensors; out_h has hit_idx, n_hits, qop, chi2, status[2], n_hits_total[1]."""
        vs = velo_states(velo_h[0].data_ptr(), velo_h[1].data_ptr(), velo_h[2].data_ptr(), velo_h[3].data_ptr(),
                         float(velo_z))
        tr = ut_tracks(out_h["hit_idx"].data_ptr(), out_h["n_hits"].data_ptr(), out_h["qop"].data_ptr(),
                       out_h["chi2"].data_ptr(), None)
        _check(_lib.ut_pipeline_run_host(self.h, raw_h.data_ptr(), raw_bytes, bank_offsets_h.data_ptr(), C.byref(vs),
                                         velo_offsets_h.data_ptr(), n_velo, n_events, C.byref(config), C.byref(tr),
                                         out_h["status"].data_ptr(), out_h["n_hits_total"].data_ptr(),
                                         _stream_ptr(stream)), "ut_pipeline_run_host")

    def timeline(self) -> list:
        """Per chunk of the last run_host (after a sync): ms from the call's start to copy-in, VELO-in, decoded, tracked, out."""
        ms = (C.c_float * 20)()
        n = C.c_int32(0)
        _check(_lib.ut_pipeline_timeline(self.h, ms, C.byref(n)), "ut_pipeline_timeline")
        keys = ("banks_in", "velo_in", "decoded", "tracked", "tracks_out")
        return [{k: round(float(ms[c * 5 + q]), 4) for q, k in enumerate(keys)} for c in range(n.value)]

    def destroy(self):
        if self.h:
            _lib.ut_pipeline_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
