"""ctypes binding of ``libtpc_tracker.so`` (include/tpc_tracker.h) - argument marshalling only.

PyTorch is used for device memory and streams; nothing here computes.
"""
from __future__ import annotations

import ctypes as C
import os
import re
from dataclasses import dataclass, fields
from typing import Dict, List, Optional

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(HERE, "libtpc_tracker.so")
_HEADER = os.path.join(os.path.dirname(HERE), "include", "tpc_tracker.h")

STATUS_TRACKLET_OVERFLOW, STATUS_TRACK_OVERFLOW, STATUS_HIT_OVERFLOW = 1, 2, 4
COUNTER_NAMES = ["clusters", "bins", "start_hits", "tracklets_built", "tracklets_kept", "chain_hits", "searches",
                 "candidates", "tracklet_hits", "row_steps", "nf_pairs", "unused", "searches_up", "candidates_up",
                 "refit_steps", "unused2"]


class TpcError(RuntimeError):
    pass


class _Geometry(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", C.POINTER(C.c_float)),
                ("tan_half_angle", C.c_float), ("z_max", C.c_float)]


_PARAM_FLOATS = ("sigma_y", "sigma_z", "nf_hy", "nf_hz", "nf_chi2_max", "grid_bin_min", "grid_bin_max", "max_sinphi",
                 "c0_sinphi", "c0_dzds", "c0_qpt", "accept_k2", "search_max", "turn_cov_scale")
_PARAM_INTS = ("min_seed_hits", "max_row_gap", "min_track_hits", "nf_z_projection")


class _Params(C.Structure):
    _fields_ = [(n, C.c_float) for n in _PARAM_FLOATS] + [(n, C.c_int32) for n in _PARAM_INTS]


class _Clusters(C.Structure):
    _fields_ = [("x", C.c_void_p), ("y", C.c_void_p), ("z", C.c_void_p), ("charge", C.c_void_p),
                ("row_offsets", C.c_void_p), ("n_clusters", C.c_uint32), ("n_tasks", C.c_uint32)]


class _Tracks(C.Structure):
    _fields_ = [("track_capacity", C.c_uint32), ("hit_capacity", C.c_uint32), ("header", C.c_void_p),
                ("track_task", C.c_void_p), ("track_hit_begin", C.c_void_p), ("track_nhits", C.c_void_p),
                ("track_ndf", C.c_void_p), ("track_x", C.c_void_p), ("track_par", C.c_void_p),
                ("track_cov", C.c_void_p), ("track_chi2", C.c_void_p), ("hit_cluster", C.c_void_p),
                ("dbg_link_up", C.c_void_p), ("dbg_link_dn", C.c_void_p), ("dbg_clean_up", C.c_void_p),
                ("dbg_clean_dn", C.c_void_p), ("dbg_start_hits", C.c_void_p), ("dbg_n_start_hits", C.c_void_p),
                ("dbg_tracklet_capacity", C.c_uint32), ("dbg_tracklet_start", C.c_void_p),
                ("dbg_tracklet_nhits", C.c_void_p), ("dbg_tracklet_map", C.c_void_p),
                ("dbg_tracklet_par", C.c_void_p)]


@dataclass
class TrackerParams:
    """tpc_params; the defaults come from the library (tpc_default_params), not from here."""
    sigma_y: Optional[float] = None
    sigma_z: Optional[float] = None
    nf_hy: Optional[float] = None
    nf_hz: Optional[float] = None
    nf_chi2_max: Optional[float] = None
    grid_bin_min: Optional[float] = None
    grid_bin_max: Optional[float] = None
    max_sinphi: Optional[float] = None
    c0_sinphi: Optional[float] = None
    c0_dzds: Optional[float] = None
    c0_qpt: Optional[float] = None
    accept_k2: Optional[float] = None
    search_max: Optional[float] = None
    turn_cov_scale: Optional[float] = None
    min_seed_hits: Optional[int] = None
    max_row_gap: Optional[int] = None
    min_track_hits: Optional[int] = None
    nf_z_projection: Optional[int] = None


def library_path() -> str:
    return _LIB_PATH


def exported_symbols() -> List[str]:
    """Function names declared in include/tpc_tracker.h (parsed from the header text)."""
    text = open(_HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tpc_[a-z_]+)\s*\(", text)))


_lib = None


def load_library():
    """Loads the in-tree extension; raises (never falls back) when it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise TpcError(f"{_LIB_PATH} is missing: run `python -m paper_1712_09434_b200.build` "
                       "(there is no CPU fallback)")
    lib = C.CDLL(_LIB_PATH)
    vp, u32, u64p = C.c_void_p, C.c_uint32, C.POINTER(C.c_uint64)
    lib.tpc_tracker_create.restype = C.c_int
    lib.tpc_tracker_create.argtypes = [C.POINTER(_Geometry), C.c_float, C.POINTER(_Params), C.POINTER(vp)]
    lib.tpc_tracker_destroy.restype = None
    lib.tpc_tracker_destroy.argtypes = [vp]
    lib.tpc_default_params.restype = None
    lib.tpc_default_params.argtypes = [C.POINTER(_Params)]
    lib.tpc_workspace_bytes.restype = C.c_size_t
    lib.tpc_workspace_bytes.argtypes = [vp, u32, u32, u32]
    lib.tpc_host_workspace_bytes.restype = C.c_size_t
    lib.tpc_host_workspace_bytes.argtypes = [vp, u32, u32, u32, u32, u32]
    lib.tpc_track_batch.restype = C.c_int
    lib.tpc_track_batch.argtypes = [vp, C.POINTER(_Clusters), C.POINTER(_Tracks), vp, C.c_size_t, u32, vp]
    lib.tpc_track_batch_host.restype = C.c_int
    lib.tpc_track_batch_host.argtypes = [vp, C.POINTER(_Clusters), C.POINTER(_Tracks), vp, C.c_size_t, u32, vp,
                                         u64p, u64p]
    lib.tpc_tracker_enable_counters.restype = None
    lib.tpc_tracker_enable_counters.argtypes = [vp, C.c_int]
    lib.tpc_read_counters.restype = C.c_int
    lib.tpc_read_counters.argtypes = [vp, vp, u64p]
    lib.tpc_launches_per_batch.restype = C.c_int
    lib.tpc_launches_per_batch.argtypes = [vp]
    lib.tpc_tracker_enable_stage_timing.restype = None
    lib.tpc_tracker_enable_stage_timing.argtypes = [vp, C.c_int]
    lib.tpc_read_stage_ms.restype = C.c_int
    lib.tpc_read_stage_ms.argtypes = [vp, vp, C.POINTER(C.c_float), C.POINTER(C.c_uint32)]
    lib.tpc_stage_name.restype = C.c_char_p
    lib.tpc_stage_name.argtypes = [C.c_int]
    lib.tpc_last_error.restype = C.c_char_p
    lib.tpc_last_error.argtypes = [vp]
    lib.tpc_host_submit.restype = C.c_int
    lib.tpc_host_submit.argtypes = [vp, C.c_int, C.POINTER(_Clusters), C.c_uint32, C.c_uint32, vp, C.c_size_t, C.c_uint32]
    lib.tpc_host_collect.restype = C.c_int
    lib.tpc_host_collect.argtypes = [vp, C.c_int, C.POINTER(_Tracks), C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    lib.tpc_its_default_params.restype = None
    lib.tpc_its_default_params.argtypes = [C.POINTER(_ItsParams)]
    lib.tpc_its_create.restype = C.c_int
    lib.tpc_its_create.argtypes = [C.POINTER(_ItsGeometry), C.c_float, C.POINTER(_ItsParams), C.POINTER(vp)]
    lib.tpc_its_destroy.restype = None
    lib.tpc_its_destroy.argtypes = [vp]
    lib.tpc_its_workspace_bytes.restype = C.c_size_t
    lib.tpc_its_workspace_bytes.argtypes = [vp, C.c_uint32, C.c_uint32]
    lib.tpc_its_track_batch.restype = C.c_int
    lib.tpc_its_track_batch.argtypes = [vp, vp, vp, vp, vp, vp, C.c_uint32, C.c_uint32, C.POINTER(_ItsTracks), vp,
                                        C.c_size_t, vp]
    lib.tpc_its_last_error.restype = C.c_char_p
    lib.tpc_its_last_error.argtypes = [vp]
    lib.tpc_slice_workspace_bytes.restype = C.c_size_t
    lib.tpc_slice_workspace_bytes.argtypes = [C.c_uint32, C.c_int32, C.c_int32]
    lib.tpc_slice_static_setup.restype = C.c_int
    lib.tpc_slice_static_setup.argtypes = []
    lib.tpc_slice_frames_static.restype = C.c_int
    lib.tpc_slice_frames_static.argtypes = [vp, vp, vp, C.c_uint32, C.c_uint32, C.c_int32, C.c_int32, C.c_float, C.c_int32,
                                            vp, vp, vp, vp, vp]
    lib.tpc_slice_frames.restype = C.c_int
    lib.tpc_slice_frames.argtypes = [vp, vp, vp, C.c_uint32, C.c_uint32, C.c_int32, C.c_int32, C.c_float, C.c_int32,
                                     vp, vp, vp, vp, vp, C.c_size_t, vp]
    lib.tpc_transform_create.restype = C.c_int
    lib.tpc_transform_create.argtypes = [C.POINTER(_Geometry), C.POINTER(_Calibration), C.POINTER(vp)]
    lib.tpc_transform_destroy.restype = None
    lib.tpc_transform_destroy.argtypes = [vp]
    lib.tpc_transform_clusters.restype = C.c_int
    lib.tpc_transform_clusters.argtypes = [vp, vp, vp, vp, C.c_uint32, C.c_uint32, vp, vp, vp]
    lib.tpc_transform_last_error.restype = C.c_char_p
    lib.tpc_transform_last_error.argtypes = [vp]
    lib.tpc_default_merge_params.restype = None
    lib.tpc_default_merge_params.argtypes = [C.POINTER(_MergeParams)]
    lib.tpc_merge_workspace_bytes.restype = C.c_size_t
    lib.tpc_merge_workspace_bytes.argtypes = [vp, C.c_uint32, C.c_uint32]
    lib.tpc_merge_refit.restype = C.c_int
    lib.tpc_merge_refit.argtypes = [vp, C.POINTER(_Clusters), C.POINTER(_Tracks), C.POINTER(_MergeParams),
                                    C.POINTER(_Merged), vp, C.c_size_t, C.c_uint32, vp, C.c_size_t, vp]
    _lib = lib
    return lib


class _Calibration(C.Structure):
    _fields_ = [("pad_pitch", C.POINTER(C.c_float)), ("n_pads", C.POINTER(C.c_int32)), ("t0", C.c_float),
                ("v_drift", C.c_float), ("t_max", C.c_float), ("map_ny", C.c_int32), ("map_nz", C.c_int32),
                ("map", C.POINTER(C.c_float))]


class _ItsGeometry(C.Structure):
    _fields_ = [("R", C.c_float * 6), ("sig_rphi", C.c_float * 6), ("sig_z", C.c_float * 6), ("xx0", C.c_float * 6)]


_ITS_FLOATS = ("max_sinphi_pair", "max_dtan", "sig_sinphi", "sig_tan", "sig_vtx_xy", "sig_vtx_z", "chi2_max", "max_dx",
               "c0_sinphi", "c0_dzds", "c0_qpt", "turn_cov_scale", "max_sinphi")


class _ItsParams(C.Structure):
    _fields_ = [(n, C.c_float) for n in _ITS_FLOATS] + [("min_clusters", C.c_int32)]


class _ItsTracks(C.Structure):
    _fields_ = [("capacity", C.c_uint32)] + [(n, C.c_void_p) for n in (
        "header", "event", "cluster", "n_clusters", "frame", "out_state", "in_state", "out_ndf", "in_ndf")]


class _MergeParams(C.Structure):
    _fields_ = [("merge_chi2_max", C.c_float), ("merge_max_row_gap", C.c_int32), ("n_slices", C.c_int32)]


class _Merged(C.Structure):
    _fields_ = [("capacity", C.c_uint32)] + [(n, C.c_void_p) for n in (
        "header", "seg_next", "seg_prev", "merged_first", "merged_nseg", "merged_nhits", "merged_nfit",
        "merged_sector", "merged_ndf", "merged_x", "merged_par", "merged_cov", "merged_chi2")]


@dataclass
class MergedResult:
    """Device tensors of one tpc_merge_refit call; sizes are capacities."""
    header: "object"
    seg_next: "object"
    seg_prev: "object"
    merged_first: "object"
    merged_nseg: "object"
    merged_nhits: "object"
    merged_nfit: "object"
    merged_sector: "object"
    merged_ndf: "object"
    merged_x: "object"
    merged_par: "object"   # [5, capacity]
    merged_cov: "object"   # [15, capacity]
    merged_chi2: "object"

    def to_numpy(self, n_tracks: int) -> Dict[str, np.ndarray]:
        """Copies to host and trims to the counts (synchronises); n_tracks = sector tracks of the tracker's call."""
        h = self.header.cpu().numpy().astype(np.int64)
        nm = int(min(h[0], self.merged_first.shape[0]))
        out = {"n_merged": int(h[0]), "n_links": int(h[1]), "status": int(h[2])}
        for f in ("seg_next", "seg_prev"):
            out[f] = getattr(self, f)[:n_tracks].cpu().numpy()
        for f in ("merged_first", "merged_nseg", "merged_nhits", "merged_nfit", "merged_sector", "merged_ndf",
                  "merged_x", "merged_chi2"):
            out[f] = getattr(self, f)[:nm].cpu().numpy()
        out["merged_par"] = self.merged_par[:, :nm].cpu().numpy()
        out["merged_cov"] = self.merged_cov[:, :nm].cpu().numpy()
        return out


@dataclass
class TrackResult:
    """Device (or pinned host) tensors of one tpc_track_batch call; sizes are capacities."""
    header: "object"
    track_task: "object"
    track_hit_begin: "object"
    track_nhits: "object"
    track_ndf: "object"
    track_x: "object"
    track_par: "object"   # [5, track_capacity]
    track_cov: "object"   # [15, track_capacity]
    track_chi2: "object"
    hit_cluster: "object"
    debug: Dict[str, "object"]

    def to_numpy(self) -> Dict[str, np.ndarray]:
        """Copies to host and trims to header counts (synchronises)."""
        h = self.header.cpu().numpy().astype(np.int64)
        nt, nh = int(min(h[0], self.track_task.shape[0])), int(min(h[1], self.hit_cluster.shape[0]))
        out = {"n_tracks": int(h[0]), "n_hits": int(h[1]), "status": int(h[2]), "n_tracklets": int(h[3])}
        for f in ("track_task", "track_hit_begin", "track_nhits", "track_ndf", "track_x", "track_chi2"):
            out[f] = getattr(self, f)[:nt].cpu().numpy()
        out["track_par"] = self.track_par[:, :nt].cpu().numpy()
        out["track_cov"] = self.track_cov[:, :nt].cpu().numpy()
        out["hit_cluster"] = self.hit_cluster[:nh].cpu().numpy()
        for k, v in self.debug.items():
            out[k] = v.cpu().numpy()
        return out


class Tracker:
    """Owns one ``tpc_tracker`` handle.  ``geometry``: object with n_sectors, n_rows, row_x (fp32),
    tan_half_angle, z_max, bz_kgauss (e.g. tpc_workload.Geometry)."""

    def __init__(self, geometry, params: Optional[TrackerParams] = None, bz_kgauss: Optional[float] = None):
        self._lib = load_library()
        self._h = C.c_void_p()
        self.n_rows = int(geometry.n_rows)
        self.n_sectors = int(geometry.n_sectors)
        row_x = np.ascontiguousarray(geometry.row_x, dtype=np.float32)
        g = _Geometry(self.n_sectors, self.n_rows, row_x.ctypes.data_as(C.POINTER(C.c_float)),
                      float(geometry.tan_half_angle), float(geometry.z_max))
        p = _Params()
        self._lib.tpc_default_params(C.byref(p))
        if params is not None:
            for f in fields(params):
                v = getattr(params, f.name)
                if v is not None:
                    setattr(p, f.name, v)
        self.params = {n: getattr(p, n) for n, _ in _Params._fields_}
        bz = float(geometry.bz_kgauss if bz_kgauss is None else bz_kgauss)
        rc = self._lib.tpc_tracker_create(C.byref(g), bz, C.byref(p), C.byref(self._h))
        if rc != 0:
            raise TpcError(f"tpc_tracker_create failed ({rc}): {self._lib.tpc_last_error(None).decode()}")
        self._ws = None

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.tpc_tracker_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def _check(self, rc, what):
        if rc != 0:
            raise TpcError(f"{what} failed ({rc}): {self._lib.tpc_last_error(self._h).decode()}")

    # ---- sizes ------------------------------------------------------------
    def workspace_bytes(self, max_clusters: int, max_tasks: int, max_tracklets: int = 0) -> int:
        return int(self._lib.tpc_workspace_bytes(self._h, max_clusters, max_tasks, max_tracklets))

    def host_workspace_bytes(self, max_clusters, max_tasks, max_tracklets, track_capacity, hit_capacity) -> int:
        return int(self._lib.tpc_host_workspace_bytes(self._h, max_clusters, max_tasks, max_tracklets,
                                                      track_capacity, hit_capacity))

    def launches_per_batch(self) -> int:
        return int(self._lib.tpc_launches_per_batch(self._h))

    def enable_counters(self, on: bool):
        self._lib.tpc_tracker_enable_counters(self._h, 1 if on else 0)

    def read_counters(self, stream=None) -> Dict[str, int]:
        buf = (C.c_uint64 * len(COUNTER_NAMES))()
        self._check(self._lib.tpc_read_counters(self._h, _stream_ptr(stream), buf), "tpc_read_counters")
        return {n: int(v) for n, v in zip(COUNTER_NAMES, buf)}

    def enable_stage_timing(self, on: bool):
        self._lib.tpc_tracker_enable_stage_timing(self._h, 1 if on else 0)

    def read_stage_ms(self, stream=None):
        """({stage name: mean ms}, calls averaged) of the calls since enable_stage_timing(True); synchronises."""
        names = []
        while self._lib.tpc_stage_name(len(names)) is not None:
            names.append(self._lib.tpc_stage_name(len(names)).decode())
        buf = (C.c_float * len(names))()
        n = C.c_uint32(0)
        self._check(self._lib.tpc_read_stage_ms(self._h, _stream_ptr(stream), buf, C.byref(n)), "tpc_read_stage_ms")
        return {k: float(v) for k, v in zip(names, buf)}, int(n.value)

    # ---- allocation helpers (torch = device memory only) ---------------------
    def alloc_outputs(self, n_clusters: int, device, track_capacity: Optional[int] = None,
                      hit_capacity: Optional[int] = None, debug: bool = False, debug_tracklets: int = 0,
                      pinned_host: bool = False) -> TrackResult:
        import torch
        tcap = int(track_capacity if track_capacity is not None else n_clusters // max(self.params["min_track_hits"], 1) + 1)
        hcap = int(hit_capacity if hit_capacity is not None else n_clusters + 1)
        kw = dict(device="cpu", pin_memory=True) if pinned_host else dict(device=device)
        e = lambda shape, dt: torch.empty(shape, dtype=dt, **kw)  # noqa: E731
        dbg = {}
        if debug:
            for k in ("dbg_link_up", "dbg_link_dn", "dbg_clean_up", "dbg_clean_dn"):
                dbg[k] = e(max(n_clusters, 1), torch.int32)
            dbg["dbg_start_hits"] = e(max(n_clusters, 1), torch.int32)
            dbg["dbg_n_start_hits"] = e(1, torch.int32)
        if debug_tracklets:
            dbg["dbg_tracklet_start"] = e(debug_tracklets, torch.int32)
            dbg["dbg_tracklet_nhits"] = e(debug_tracklets, torch.int32)
            dbg["dbg_tracklet_map"] = e((debug_tracklets, self.n_rows), torch.int32)
            dbg["dbg_tracklet_par"] = e((debug_tracklets, 5), torch.float32)
        return TrackResult(
            header=e(4, torch.int32), track_task=e(tcap, torch.int32), track_hit_begin=e(tcap, torch.int32),
            track_nhits=e(tcap, torch.int32), track_ndf=e(tcap, torch.int32), track_x=e(tcap, torch.float32),
            track_par=e((5, tcap), torch.float32), track_cov=e((15, tcap), torch.float32),
            track_chi2=e(tcap, torch.float32), hit_cluster=e(hcap, torch.int32), debug=dbg)

    def alloc_workspace(self, nbytes: int, device):
        import torch
        return torch.empty(nbytes + 256, dtype=torch.uint8, device=device)

    @staticmethod
    def _aligned(ws):
        p = ws.data_ptr()
        off = (-p) % 256
        return p + off, ws.numel() - off

    def _tracks_struct(self, out: TrackResult) -> _Tracks:
        t = _Tracks()
        t.track_capacity = int(out.track_task.shape[0])
        t.hit_capacity = int(out.hit_cluster.shape[0])
        for f in ("header", "track_task", "track_hit_begin", "track_nhits", "track_ndf", "track_x", "track_par",
                  "track_cov", "track_chi2", "hit_cluster"):
            setattr(t, f, getattr(out, f).data_ptr())
        for k, v in out.debug.items():
            setattr(t, k, v.data_ptr())
        if "dbg_tracklet_start" in out.debug:
            t.dbg_tracklet_capacity = int(out.debug["dbg_tracklet_start"].shape[0])
        return t

    # ---- the two compute entry points ---------------------------------------
    def track_batch(self, y, z, row_offsets, n_tasks: int, out: TrackResult, workspace, max_tracklets: int = 0,
                    stream=None, x=None, charge=None) -> TrackResult:
        """tpc_track_batch on DEVICE tensors (y, z fp32; row_offsets int32/uint32 viewed as uint32).
        Asynchronous on ``stream`` (a torch.cuda.Stream; default: the current stream)."""
        import torch
        if not (y.is_cuda and z.is_cuda and row_offsets.is_cuda):
            raise TpcError("track_batch needs CUDA tensors; there is no CPU path")
        assert y.dtype == torch.float32 and z.dtype == torch.float32 and row_offsets.dtype == torch.int32
        assert y.is_contiguous() and z.is_contiguous() and row_offsets.is_contiguous()
        assert row_offsets.numel() == n_tasks * self.n_rows + 1
        cl = _Clusters(x.data_ptr() if x is not None else None, y.data_ptr(), z.data_ptr(),
                       charge.data_ptr() if charge is not None else None, row_offsets.data_ptr(),
                       int(y.numel()), int(n_tasks))
        tr = self._tracks_struct(out)
        wp, wn = self._aligned(workspace)
        s = stream if stream is not None else torch.cuda.current_stream(y.device)
        self._check(self._lib.tpc_track_batch(self._h, C.byref(cl), C.byref(tr), wp, wn, int(max_tracklets),
                                              _stream_ptr(s)), "tpc_track_batch")
        return out

    def track_batch_host(self, y, z, row_offsets, n_tasks: int, out: TrackResult, workspace,
                         max_tracklets: int = 0, stream=None):
        """tpc_track_batch_host on HOST tensors (pinned recommended); synchronous.
        Returns (h2d_bytes, d2h_bytes)."""
        import torch
        assert not y.is_cuda and not z.is_cuda and not row_offsets.is_cuda and workspace.is_cuda
        assert y.dtype == torch.float32 and z.dtype == torch.float32 and row_offsets.dtype == torch.int32
        cl = _Clusters(None, y.data_ptr(), z.data_ptr(), None, row_offsets.data_ptr(), int(y.numel()), int(n_tasks))
        tr = self._tracks_struct(out)
        wp, wn = self._aligned(workspace)
        s = stream if stream is not None else torch.cuda.current_stream(workspace.device)
        up, down = C.c_uint64(0), C.c_uint64(0)
        self._check(self._lib.tpc_track_batch_host(self._h, C.byref(cl), C.byref(tr), wp, wn, int(max_tracklets),
                                                   _stream_ptr(s), C.byref(up), C.byref(down)),
                    "tpc_track_batch_host")
        return int(up.value), int(down.value)


    def host_submit(self, slot: int, y, z, row_offsets, n_tasks: int, track_capacity: int, hit_capacity: int,
                    workspace, max_tracklets: int = 0):
        """tpc_host_submit: HOST tensors (pinned), returns at once; the tensors must stay alive until host_collect."""
        import torch
        assert not y.is_cuda and not z.is_cuda and not row_offsets.is_cuda and workspace.is_cuda
        assert y.dtype == torch.float32 and z.dtype == torch.float32 and row_offsets.dtype == torch.int32
        cl = _Clusters(None, y.data_ptr(), z.data_ptr(), None, row_offsets.data_ptr(), int(y.numel()), int(n_tasks))
        wp, wn = self._aligned(workspace)
        self._check(self._lib.tpc_host_submit(self._h, int(slot), C.byref(cl), int(track_capacity), int(hit_capacity),
                                              wp, wn, int(max_tracklets)), "tpc_host_submit")

    def host_collect(self, slot: int, out: TrackResult):
        """tpc_host_collect into HOST tensors; returns (h2d_bytes, d2h_bytes) of the batch."""
        tr = self._tracks_struct(out)
        up, down = C.c_uint64(0), C.c_uint64(0)
        self._check(self._lib.tpc_host_collect(self._h, int(slot), C.byref(tr), C.byref(up), C.byref(down)),
                    "tpc_host_collect")
        return int(up.value), int(down.value)

    # ---- sector-segment merger + refit (include/tpc_tracker.h, SPEC 9) ----------------------
    def merge_workspace_bytes(self, track_capacity: int, max_tasks: int) -> int:
        return int(self._lib.tpc_merge_workspace_bytes(self._h, track_capacity, max_tasks))

    def alloc_merged(self, capacity: int, device) -> "MergedResult":
        import torch
        e = lambda shape, dt: torch.empty(shape, dtype=dt, device=device)  # noqa: E731
        cap = max(int(capacity), 1)
        return MergedResult(
            header=e(4, torch.int32), seg_next=e(cap, torch.int32), seg_prev=e(cap, torch.int32),
            merged_first=e(cap, torch.int32), merged_nseg=e(cap, torch.int32), merged_nhits=e(cap, torch.int32),
            merged_nfit=e(cap, torch.int32), merged_sector=e(cap, torch.int32), merged_ndf=e(cap, torch.int32),
            merged_x=e(cap, torch.float32), merged_par=e((5, cap), torch.float32),
            merged_cov=e((15, cap), torch.float32), merged_chi2=e(cap, torch.float32))

    def merge_refit(self, y, z, row_offsets, n_tasks: int, tracks: TrackResult, merged: "MergedResult", workspace,
                    merge_workspace, max_tracklets: int = 0, chi2_max: Optional[float] = None,
                    max_row_gap: Optional[int] = None, n_slices: int = 1, stream=None) -> "MergedResult":
        """tpc_merge_refit right after track_batch with the same tensors and workspace. Asynchronous."""
        import torch
        cl = _Clusters(None, y.data_ptr(), z.data_ptr(), None, row_offsets.data_ptr(), int(y.numel()), int(n_tasks))
        tr = self._tracks_struct(tracks)
        mp = _MergeParams()
        self._lib.tpc_default_merge_params(C.byref(mp))
        if chi2_max is not None:
            mp.merge_chi2_max = chi2_max
        if max_row_gap is not None:
            mp.merge_max_row_gap = max_row_gap
        mp.n_slices = int(n_slices)
        mg = _Merged()
        mg.capacity = int(merged.seg_next.shape[0])
        for n, _ in _Merged._fields_[1:]:
            setattr(mg, n, getattr(merged, n).data_ptr())
        wp, wn = self._aligned(workspace)
        mwp, mwn = self._aligned(merge_workspace)
        s = stream if stream is not None else torch.cuda.current_stream(y.device)
        self._check(self._lib.tpc_merge_refit(self._h, C.byref(cl), C.byref(tr), C.byref(mp), C.byref(mg), wp, wn,
                                              int(max_tracklets), mwp, mwn, _stream_ptr(s)), "tpc_merge_refit")
        return merged


def slice_frames(y, zeta, row_offsets, n_tasks_in: int, n_sectors: int, n_rows: int, slice_len: float, n_slices: int,
                 stream=None):
    """tpc_slice_frames on DEVICE tensors; returns (y_out, z_out, src_index, row_offsets_out) device tensors
    (int32 views of the uint32 arrays).  Asynchronous."""
    import torch
    lib = load_library()
    if not (y.is_cuda and zeta.is_cuda and row_offsets.is_cuda):
        raise TpcError("slice_frames needs CUDA tensors; there is no CPU path")
    dev = y.device
    n = int(y.numel())
    y_out, z_out = torch.empty_like(y), torch.empty_like(zeta)
    src = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
    ro_out = torch.empty(n_tasks_in * n_slices * n_rows + 1, dtype=torch.int32, device=dev)
    wb = int(lib.tpc_slice_workspace_bytes(n_tasks_in, n_rows, n_slices))
    ws = torch.empty(wb + 256, dtype=torch.uint8, device=dev)
    wp = ws.data_ptr() + (-ws.data_ptr()) % 256
    s = stream if stream is not None else torch.cuda.current_stream(dev)
    rc = lib.tpc_slice_frames(y.data_ptr(), zeta.data_ptr(), row_offsets.data_ptr(), n, int(n_tasks_in), int(n_sectors),
                              int(n_rows), float(slice_len), int(n_slices), y_out.data_ptr(), z_out.data_ptr(),
                              src.data_ptr(), ro_out.data_ptr(), wp, wb, _stream_ptr(s))
    if rc != 0:
        raise TpcError(f"tpc_slice_frames failed ({rc}): {lib.tpc_last_error(None).decode()}")
    slice_frames._keep = ws  # the workspace must outlive the asynchronous kernels
    return y_out, z_out, src[:n], ro_out


SLICE_STATIC_MAX_ENTRIES = 1 << 20  # include/tpc_tracker.h: TPC_SLICE_STATIC_MAX_ENTRIES


def slice_static_setup():
    """tpc_slice_static_setup for the current CUDA device (once per device, at set-up)."""
    lib = load_library()
    rc = lib.tpc_slice_static_setup()
    if rc != 0:
        raise TpcError(f"tpc_slice_static_setup failed ({rc}): {lib.tpc_last_error(None).decode()}")


def slice_frames_static(y, zeta, row_offsets, n_tasks_in: int, n_sectors: int, n_rows: int, slice_len: float,
                        n_slices: int, y_out, z_out, src_index, row_offsets_out, stream=None):
    """tpc_slice_frames_static on DEVICE tensors the caller owns (inputs and outputs): the library allocates
    nothing, its scratch is a static device array shared by all calls on the device (calls that overlap on the
    GPU race).  Sizes beyond TPC_SLICE_STATIC_MAX_ENTRIES raise.  Asynchronous."""
    import torch
    lib = load_library()
    for t in (y, zeta, row_offsets, y_out, z_out, src_index, row_offsets_out):
        if not t.is_cuda:
            raise TpcError("slice_frames_static needs CUDA tensors; there is no CPU path")
    n = int(y.numel())
    if int(y_out.numel()) < n or int(z_out.numel()) < n or int(src_index.numel()) < n or \
            int(row_offsets_out.numel()) < n_tasks_in * n_slices * n_rows + 1:
        raise TpcError("slice_frames_static: an output tensor is too small")
    s = stream if stream is not None else torch.cuda.current_stream(y.device)
    with torch.cuda.device(y.device):
        rc = lib.tpc_slice_frames_static(y.data_ptr(), zeta.data_ptr(), row_offsets.data_ptr(), n, int(n_tasks_in),
                                         int(n_sectors), int(n_rows), float(slice_len), int(n_slices),
                                         y_out.data_ptr(), z_out.data_ptr(), src_index.data_ptr(),
                                         row_offsets_out.data_ptr(), _stream_ptr(s))
    if rc != 0:
        raise TpcError(f"tpc_slice_frames_static failed ({rc}): {lib.tpc_last_error(None).decode()}")


class ItsTracker:
    """Owns one ``tpc_its_tracker`` handle (SPEC 12).  ``geometry``: object with R, sig_rphi, sig_z, xx0 [6] and
    bz_kgauss (e.g. tpc_workload.ItsGeometry); ``params``: dict of tpc_its_params fields to change."""

    def __init__(self, geometry, params: Optional[dict] = None):
        self._lib = load_library()
        self._h = C.c_void_p()
        g = _ItsGeometry()
        for l in range(6):
            g.R[l], g.sig_rphi[l] = float(geometry.R[l]), float(geometry.sig_rphi[l])
            g.sig_z[l], g.xx0[l] = float(geometry.sig_z[l]), float(geometry.xx0[l])
        p = _ItsParams()
        self._lib.tpc_its_default_params(C.byref(p))
        for k, v in (params or {}).items():
            setattr(p, k, v)
        rc = self._lib.tpc_its_create(C.byref(g), float(geometry.bz_kgauss), C.byref(p), C.byref(self._h))
        if rc != 0:
            raise TpcError(f"tpc_its_create failed ({rc}): {self._lib.tpc_its_last_error(None).decode()}")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.tpc_its_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def track_batch(self, x, y, z, layer_offsets, vertex, n_events: int, capacity: Optional[int] = None, stream=None):
        """tpc_its_track_batch on DEVICE tensors; returns a dict of device tensors (header, event, cluster, ...).
        Asynchronous; the returned dict keeps the workspace alive."""
        import torch
        if not (x.is_cuda and y.is_cuda and z.is_cuda and layer_offsets.is_cuda and vertex.is_cuda):
            raise TpcError("ItsTracker.track_batch needs CUDA tensors; there is no CPU path")
        dev = x.device
        n = int(x.numel())
        cap = int(capacity if capacity is not None else n // 2 + 1)
        e = lambda shape, dt: torch.empty(shape, dtype=dt, device=dev)  # noqa: E731
        out = dict(header=e(4, torch.int32), event=e(cap, torch.int32), cluster=e((cap, 6), torch.int32),
                   n_clusters=e(cap, torch.int32), frame=e((cap, 2), torch.float32), out_state=e((cap, 22), torch.float32),
                   in_state=e((cap, 22), torch.float32), out_ndf=e(cap, torch.int32), in_ndf=e(cap, torch.int32))
        tr = _ItsTracks()
        tr.capacity = cap
        for k_, v in out.items():
            setattr(tr, k_, v.data_ptr())
        wb = int(self._lib.tpc_its_workspace_bytes(self._h, n, int(n_events)))
        ws = torch.empty(wb + 256, dtype=torch.uint8, device=dev)
        wp = ws.data_ptr() + (-ws.data_ptr()) % 256
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        rc = self._lib.tpc_its_track_batch(self._h, x.data_ptr(), y.data_ptr(), z.data_ptr(), layer_offsets.data_ptr(),
                                           vertex.data_ptr(), n, int(n_events), C.byref(tr), wp, wb, _stream_ptr(s))
        if rc != 0:
            raise TpcError(f"tpc_its_track_batch failed ({rc}): {self._lib.tpc_its_last_error(self._h).decode()}")
        out["_workspace"] = ws
        return out


class ClusterTransform:
    """Owns one ``tpc_transform`` handle (SPEC 10).  ``calibration``: object with pad_pitch, n_pads, t0, v_drift,
    t_max, corr [n_sectors, n_rows, MZ, MY, 2] (e.g. tpc_workload.RawCalibration)."""

    def __init__(self, geometry, calibration):
        self._lib = load_library()
        self._h = C.c_void_p()
        self.n_rows = int(geometry.n_rows)
        row_x = np.ascontiguousarray(geometry.row_x, dtype=np.float32)
        g = _Geometry(int(geometry.n_sectors), self.n_rows, row_x.ctypes.data_as(C.POINTER(C.c_float)),
                      float(geometry.tan_half_angle), float(geometry.z_max))
        pitch = np.ascontiguousarray(calibration.pad_pitch, np.float32)
        npads = np.ascontiguousarray(calibration.n_pads, np.int32)
        corr = np.ascontiguousarray(calibration.corr, np.float32)
        assert corr.shape[:2] == (int(geometry.n_sectors), self.n_rows) and corr.shape[4] == 2
        cal = _Calibration(pitch.ctypes.data_as(C.POINTER(C.c_float)), npads.ctypes.data_as(C.POINTER(C.c_int32)),
                           float(calibration.t0), float(calibration.v_drift), float(calibration.t_max),
                           int(corr.shape[3]), int(corr.shape[2]), corr.ctypes.data_as(C.POINTER(C.c_float)))
        rc = self._lib.tpc_transform_create(C.byref(g), C.byref(cal), C.byref(self._h))
        if rc != 0:
            raise TpcError(f"tpc_transform_create failed ({rc}): {self._lib.tpc_transform_last_error(None).decode()}")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.tpc_transform_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def transform(self, pad, time, row_offsets, n_tasks: int, y, z, stream=None):
        """tpc_transform_clusters on DEVICE tensors (fp32; row_offsets int32 viewed as uint32). Asynchronous."""
        import torch
        if not (pad.is_cuda and time.is_cuda and row_offsets.is_cuda and y.is_cuda and z.is_cuda):
            raise TpcError("transform needs CUDA tensors; there is no CPU path")
        assert pad.dtype == time.dtype == y.dtype == z.dtype == torch.float32 and row_offsets.dtype == torch.int32
        assert row_offsets.numel() == n_tasks * self.n_rows + 1 and y.numel() == z.numel() == pad.numel() == time.numel()
        s = stream if stream is not None else torch.cuda.current_stream(pad.device)
        rc = self._lib.tpc_transform_clusters(self._h, pad.data_ptr(), time.data_ptr(), row_offsets.data_ptr(),
                                              int(pad.numel()), int(n_tasks), y.data_ptr(), z.data_ptr(), _stream_ptr(s))
        if rc != 0:
            raise TpcError(f"tpc_transform_clusters failed ({rc}): {self._lib.tpc_transform_last_error(self._h).decode()}")


def _stream_ptr(stream):
    if stream is None:
        return None
    return C.c_void_p(int(stream.cuda_stream))
