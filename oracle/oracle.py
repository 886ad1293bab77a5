"""ctypes wrapper of ``libtpc_oracle.so`` (CPU oracle, test infrastructure).

Nothing here does tracker arithmetic: it marshals numpy arrays into the C++
oracle (``tpc_oracle.cpp``) and back.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass, field
from typing import Dict, Optional

import numpy as np

from . import build as _build

COUNTER_NAMES = [
    "clusters", "bins", "nf_pairs", "start_hits", "tracklets_built", "tracklets_kept", "chain_hits",
    "search_up", "search_dn", "candidates", "tracklet_hits", "out_hits", "out_tracks", "row_steps",
]


class _Geom(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", C.POINTER(C.c_float)),
                ("tan_half_angle", C.c_float), ("z_max", C.c_float)]


class _Params(C.Structure):
    _fields_ = [(n, C.c_float) for n in (
        "sigma_y", "sigma_z", "nf_hy", "nf_hz", "nf_chi2_max", "grid_bin_min", "grid_bin_max",
        "max_sinphi", "c0_sinphi", "c0_dzds", "c0_qpt", "accept_k2", "search_max", "turn_cov_scale")] + [
        (n, C.c_int32) for n in ("min_seed_hits", "max_row_gap", "min_track_hits", "nf_z_projection")]


class _Out(C.Structure):
    _fields_ = [
        ("link_up", C.c_void_p), ("link_dn", C.c_void_p), ("clean_up", C.c_void_p), ("clean_dn", C.c_void_p),
        ("start_hits", C.c_void_p),
        ("track_capacity", C.c_uint32), ("hit_capacity", C.c_uint32),
        ("track_task", C.c_void_p), ("track_hit_begin", C.c_void_p), ("track_nhits", C.c_void_p),
        ("track_ndf", C.c_void_p),
        ("track_x", C.c_void_p), ("track_par", C.c_void_p), ("track_cov", C.c_void_p), ("track_chi2", C.c_void_p),
        ("hit_cluster", C.c_void_p),
        ("tracklet_capacity", C.c_uint32),
        ("tracklet_start", C.c_void_p), ("tracklet_nhits", C.c_void_p), ("tracklet_map", C.c_void_p),
        ("tracklet_par", C.c_void_p),
        ("counters", C.c_void_p),
        ("n_start_hits", C.c_uint32), ("n_tracklets", C.c_uint32), ("n_tracks", C.c_uint32), ("n_hits", C.c_uint32),
    ]


class _MergeIn(C.Structure):
    _fields_ = [("n_tracks", C.c_uint32), ("track_capacity", C.c_uint32),
                ("track_task", C.c_void_p), ("track_hit_begin", C.c_void_p), ("track_nhits", C.c_void_p),
                ("track_ndf", C.c_void_p),
                ("track_x", C.c_void_p), ("track_par", C.c_void_p), ("track_cov", C.c_void_p),
                ("track_chi2", C.c_void_p), ("hit_cluster", C.c_void_p)]


class _MergeOut(C.Structure):
    _fields_ = [("next", C.c_void_p), ("prev", C.c_void_p), ("merged_capacity", C.c_uint32),
                ("merged_first", C.c_void_p), ("merged_nseg", C.c_void_p), ("merged_nhits", C.c_void_p),
                ("merged_nfit", C.c_void_p), ("merged_sector", C.c_void_p), ("merged_ndf", C.c_void_p),
                ("merged_x", C.c_void_p), ("merged_par", C.c_void_p), ("merged_cov", C.c_void_p),
                ("merged_chi2", C.c_void_p), ("n_merged", C.c_uint32), ("n_links", C.c_uint32)]


@dataclass
class OracleParams:
    """Defaults of docs/ARITH_SPEC.md section 8 (the oracle's own copy)."""
    sigma_y: float = 0.1
    sigma_z: float = 0.15
    nf_hy: float = 2.0
    nf_hz: float = 1.5
    nf_chi2_max: float = 75.0
    grid_bin_min: float = 2.0
    grid_bin_max: float = 20.0
    max_sinphi: float = 0.95
    c0_sinphi: float = 1.0
    c0_dzds: float = 1.0
    c0_qpt: float = 100.0
    accept_k2: float = 16.0
    search_max: float = 3.0
    turn_cov_scale: float = 100.0
    min_seed_hits: int = 5
    max_row_gap: int = 4
    min_track_hits: int = 10
    nf_z_projection: int = 1   # SPEC 11: 0 in time-frame mode

    def _c(self) -> _Params:
        return _Params(**{n: getattr(self, n) for n, _ in _Params._fields_})


@dataclass
class OracleResult:
    link_up: np.ndarray
    link_dn: np.ndarray
    clean_up: np.ndarray
    clean_dn: np.ndarray
    start_hits: np.ndarray
    track_task: np.ndarray
    track_hit_begin: np.ndarray
    track_nhits: np.ndarray
    track_ndf: np.ndarray
    track_x: np.ndarray
    track_par: np.ndarray   # [5, n_tracks]
    track_cov: np.ndarray   # [15, n_tracks]
    track_chi2: np.ndarray
    hit_cluster: np.ndarray
    counters: Dict[str, int] = field(default_factory=dict)
    n_tracklets: int = 0
    tracklet_start: Optional[np.ndarray] = None
    tracklet_nhits: Optional[np.ndarray] = None
    tracklet_map: Optional[np.ndarray] = None
    tracklet_par: Optional[np.ndarray] = None

    @property
    def n_tracks(self) -> int:
        return int(self.track_task.shape[0])

    def track_hits(self, t: int) -> np.ndarray:
        b = int(self.track_hit_begin[t])
        return self.hit_cluster[b:b + int(self.track_nhits[t])]


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_n_counters.restype = C.c_int
        _lib.oracle_sizeof_out.restype = C.c_size_t
        assert _lib.oracle_n_counters() == len(COUNTER_NAMES)
        assert _lib.oracle_sizeof_out() == C.sizeof(_Out)
        for n in ("oracle_track_f32", "oracle_track_f64"):
            getattr(_lib, n).restype = C.c_int
        _lib.oracle_transport_f64.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        _lib.oracle_transport_f32.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_float]
        _lib.oracle_update_f64.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_double]
        _lib.oracle_update_f32.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_float, C.c_float]
        _lib.oracle_sizeof_merge_in.restype = C.c_size_t
        _lib.oracle_sizeof_merge_out.restype = C.c_size_t
        assert _lib.oracle_sizeof_merge_in() == C.sizeof(_MergeIn)
        assert _lib.oracle_sizeof_merge_out() == C.sizeof(_MergeOut)
        for n in ("oracle_merge_f32", "oracle_merge_f64", "oracle_rotate_f32", "oracle_rotate_f64",
                  "oracle_refit_hits_f64"):
            getattr(_lib, n).restype = C.c_int
        _lib.oracle_rotate_f64.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double]
        _lib.oracle_rotate_f32.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_float]
    return _lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def track(geometry, y, z, row_offsets, n_tasks: int, params: Optional[OracleParams] = None,
          precision: str = "f32", brute_force_neighbours: bool = False,
          dump_tracklets: bool = False) -> OracleResult:
    """Run the whole oracle path on host arrays.

    ``geometry`` is any object with n_sectors, n_rows, row_x (fp32), tan_half_angle,
    z_max, bz_kgauss.  ``precision`` "f32" is the parity arithmetic; "f64" is the
    same sequence in double (accuracy pins only).
    """
    lib = _load()
    prm = params or OracleParams()
    dt = np.float32 if precision == "f32" else np.float64
    y = np.ascontiguousarray(y, dtype=dt)
    z = np.ascontiguousarray(z, dtype=dt)
    ro = np.ascontiguousarray(row_offsets, dtype=np.uint32)
    n = int(y.shape[0])
    nr = int(geometry.n_rows)
    assert ro.shape[0] == n_tasks * nr + 1 and int(ro[-1]) == n
    row_x = np.ascontiguousarray(geometry.row_x, dtype=np.float32)
    g = _Geom(int(geometry.n_sectors), nr, row_x.ctypes.data_as(C.POINTER(C.c_float)),
              float(geometry.tan_half_angle), float(geometry.z_max))
    tcap = n // max(prm.min_track_hits, 1) + 1
    hcap = n + 1
    i32 = lambda m: np.empty(m, np.int32)  # noqa: E731
    u32 = lambda m: np.empty(m, np.uint32)  # noqa: E731
    link_up, link_dn, clean_up, clean_dn = i32(n), i32(n), i32(n), i32(n)
    start = u32(n)
    t_task, t_beg, t_nh, t_ndf = u32(tcap), u32(tcap), u32(tcap), i32(tcap)
    t_x, t_chi2 = np.empty(tcap, dt), np.empty(tcap, dt)
    t_par, t_cov = np.empty((5, tcap), dt), np.empty((15, tcap), dt)
    hits = u32(hcap)
    counters = np.zeros(len(COUNTER_NAMES), np.uint64)
    kcap = n // 2 + 1 if dump_tracklets else 0
    k_start = u32(kcap) if dump_tracklets else None
    k_nh = u32(kcap) if dump_tracklets else None
    k_map = np.empty((kcap, nr), np.int32) if dump_tracklets else None
    k_par = np.empty((kcap, 5), dt) if dump_tracklets else None
    o = _Out(_ptr(link_up), _ptr(link_dn), _ptr(clean_up), _ptr(clean_dn), _ptr(start), tcap, hcap,
             _ptr(t_task), _ptr(t_beg), _ptr(t_nh), _ptr(t_ndf), _ptr(t_x), _ptr(t_par), _ptr(t_cov),
             _ptr(t_chi2), _ptr(hits), kcap, _ptr(k_start), _ptr(k_nh), _ptr(k_map), _ptr(k_par),
             _ptr(counters), 0, 0, 0, 0)
    fn = lib.oracle_track_f32 if precision == "f32" else lib.oracle_track_f64
    rc = fn(C.byref(g), C.c_float(float(geometry.bz_kgauss)), C.byref(prm._c()), C.c_uint32(n),
            C.c_uint32(n_tasks), _ptr(y), _ptr(z), _ptr(ro), C.byref(o), C.c_int(0 if brute_force_neighbours else 1))
    if rc != 0:
        raise RuntimeError(f"oracle_track returned {rc} (output capacity)")
    nt, nh, ns, nk = o.n_tracks, o.n_hits, o.n_start_hits, o.n_tracklets
    res = OracleResult(
        link_up, link_dn, clean_up, clean_dn, start[:ns].copy(),
        t_task[:nt].copy(), t_beg[:nt].copy(), t_nh[:nt].copy(), t_ndf[:nt].copy(), t_x[:nt].copy(),
        t_par[:, :nt].copy(), t_cov[:, :nt].copy(), t_chi2[:nt].copy(), hits[:nh].copy(),
        counters={k: int(v) for k, v in zip(COUNTER_NAMES, counters)}, n_tracklets=nk)
    if dump_tracklets:
        res.tracklet_start, res.tracklet_nhits = k_start[:nk].copy(), k_nh[:nk].copy()
        res.tracklet_map, res.tracklet_par = k_map[:nk].copy(), k_par[:nk].copy()
    return res


def transport(x, p, c, xnew, a, max_sinphi=0.95, precision="f64"):
    """SPEC 5.1 on one state; returns (ok, x, p[5], c[15])."""
    lib = _load()
    dt = np.float64 if precision == "f64" else np.float32
    s = np.zeros(22, dt)
    s[0] = x
    s[1:6] = p
    s[6:21] = c
    fn = lib.oracle_transport_f64 if precision == "f64" else lib.oracle_transport_f32
    ok = fn(_ptr(s), xnew, a, max_sinphi)
    return bool(ok), dt(s[0]), s[1:6].copy(), s[6:21].copy()


def update(p, c, i, m, e, chi2=0.0, ndf=0, precision="f64"):
    """SPEC 5.2 on one state; returns (p[5], c[15], chi2, ndf)."""
    lib = _load()
    dt = np.float64 if precision == "f64" else np.float32
    s = np.zeros(22, dt)
    s[1:6] = p
    s[6:21] = c
    s[21] = chi2
    nd = np.array([ndf], np.int32)
    fn = lib.oracle_update_f64 if precision == "f64" else lib.oracle_update_f32
    fn(_ptr(s), _ptr(nd), i, m, e)
    return s[1:6].copy(), s[6:21].copy(), dt(s[21]), int(nd[0])


@dataclass
class MergeResult:
    """SPEC 9: links between the sector tracks (G6) and the refitted merged tracks (F3)."""
    next: np.ndarray          # [n_tracks] index of the segment that continues track i outwards, or -1
    prev: np.ndarray
    merged_first: np.ndarray  # [n_merged] innermost segment (track index); merged tracks in this order
    merged_nseg: np.ndarray
    merged_nhits: np.ndarray
    merged_nfit: np.ndarray
    merged_sector: np.ndarray
    merged_ndf: np.ndarray
    merged_x: np.ndarray
    merged_par: np.ndarray    # [5, n_merged]
    merged_cov: np.ndarray    # [15, n_merged]
    merged_chi2: np.ndarray
    n_links: int = 0


def merge_refit(geometry, y, z, row_offsets, n_tasks: int, tracks, params: Optional[OracleParams] = None,
                chi2_max: float = 50.0, max_row_gap: int = 8, precision: str = "f32", n_slices: int = 1) -> MergeResult:
    """SPEC 9 on the tracks of ``track()`` (any object with track_task, track_hit_begin, track_nhits, track_x,
    track_par [5,n], track_cov [15,n], hit_cluster); the tracks may be given in any order."""
    lib = _load()
    prm = params or OracleParams()
    dt = np.float32 if precision == "f32" else np.float64
    y = np.ascontiguousarray(y, dtype=dt)
    z = np.ascontiguousarray(z, dtype=dt)
    ro = np.ascontiguousarray(row_offsets, dtype=np.uint32)
    n, nr = int(y.shape[0]), int(geometry.n_rows)
    row_x = np.ascontiguousarray(geometry.row_x, dtype=np.float32)
    g = _Geom(int(geometry.n_sectors), nr, row_x.ctypes.data_as(C.POINTER(C.c_float)),
              float(geometry.tan_half_angle), float(geometry.z_max))
    nt = int(len(tracks.track_task))
    cap = max(nt, 1)
    t_task = np.ascontiguousarray(tracks.track_task, np.uint32)
    t_beg = np.ascontiguousarray(tracks.track_hit_begin, np.uint32)
    t_nh = np.ascontiguousarray(tracks.track_nhits, np.uint32)
    t_x = np.ascontiguousarray(tracks.track_x, dt)
    t_ndf = np.ascontiguousarray(getattr(tracks, "track_ndf", np.zeros(nt)), np.int32)
    t_chi2 = np.ascontiguousarray(getattr(tracks, "track_chi2", np.zeros(nt)), dt)
    t_par = np.zeros((5, cap), dt); t_par[:, :nt] = tracks.track_par
    t_cov = np.zeros((15, cap), dt); t_cov[:, :nt] = tracks.track_cov
    hits = np.ascontiguousarray(tracks.hit_cluster, np.uint32)
    mi = _MergeIn(nt, cap, _ptr(t_task), _ptr(t_beg), _ptr(t_nh), _ptr(t_ndf), _ptr(t_x), _ptr(t_par), _ptr(t_cov),
                  _ptr(t_chi2), _ptr(hits))
    nxt, prv = np.empty(cap, np.int32), np.empty(cap, np.int32)
    u32 = lambda: np.empty(cap, np.uint32)  # noqa: E731
    m_first, m_nseg, m_nh, m_nfit, m_sec = u32(), u32(), u32(), u32(), u32()
    m_ndf = np.empty(cap, np.int32)
    m_x, m_chi2 = np.empty(cap, dt), np.empty(cap, dt)
    m_par, m_cov = np.empty((5, cap), dt), np.empty((15, cap), dt)
    mo = _MergeOut(_ptr(nxt), _ptr(prv), cap, _ptr(m_first), _ptr(m_nseg), _ptr(m_nh), _ptr(m_nfit), _ptr(m_sec),
                   _ptr(m_ndf), _ptr(m_x), _ptr(m_par), _ptr(m_cov), _ptr(m_chi2), 0, 0)
    fn = lib.oracle_merge_f32 if precision == "f32" else lib.oracle_merge_f64
    rc = fn(C.byref(g), C.c_float(float(geometry.bz_kgauss)), C.byref(prm._c()), C.c_float(chi2_max),
            C.c_int32(max_row_gap), C.c_int32(n_slices), C.c_uint32(n), C.c_uint32(n_tasks), _ptr(y), _ptr(z), _ptr(ro),
            C.byref(mi), C.byref(mo))
    if rc != 0:
        raise RuntimeError(f"oracle_merge returned {rc}")
    m = mo.n_merged
    return MergeResult(nxt[:nt].copy(), prv[:nt].copy(), m_first[:m].copy(), m_nseg[:m].copy(), m_nh[:m].copy(),
                       m_nfit[:m].copy(), m_sec[:m].copy(), m_ndf[:m].copy(), m_x[:m].copy(), m_par[:, :m].copy(),
                       m_cov[:, :m].copy(), m_chi2[:m].copy(), n_links=int(mo.n_links))


def rotate(x, p, c, d, n_sectors, a, max_sinphi=0.95, precision="f64"):
    """SPEC 9.1 on one state; returns (ok, x, p[5], c[15])."""
    lib = _load()
    dt = np.float64 if precision == "f64" else np.float32
    s = np.zeros(22, dt)
    s[0] = x
    s[1:6] = p
    s[6:21] = c
    fn = lib.oracle_rotate_f64 if precision == "f64" else lib.oracle_rotate_f32
    ok = fn(_ptr(s), int(d), int(n_sectors), a, max_sinphi)
    return bool(ok), dt(s[0]), s[1:6].copy(), s[6:21].copy()


def refit_hits(geometry, sector, row, y, z, x0, p0, c0, sector0, params: Optional[OracleParams] = None):
    """SPEC 9.3 (fp64) on an explicit hit list, outermost first, started from the state (x0, p0[5], c0[15]) in the
    frame of sector0; returns (n_fit, x, p[5], c[15], chi2, ndf, sector)."""
    lib = _load()
    prm = params or OracleParams()
    row_x = np.ascontiguousarray(geometry.row_x, dtype=np.float32)
    g = _Geom(int(geometry.n_sectors), int(geometry.n_rows), row_x.ctypes.data_as(C.POINTER(C.c_float)),
              float(geometry.tan_half_angle), float(geometry.z_max))
    sector = np.ascontiguousarray(sector, np.int32)
    row = np.ascontiguousarray(row, np.int32)
    y = np.ascontiguousarray(y, np.float64)
    z = np.ascontiguousarray(z, np.float64)
    s = np.zeros(22, np.float64)
    s[0] = x0
    s[1:6] = p0
    s[6:21] = c0
    ndf, sec = np.zeros(1, np.int32), np.array([sector0], np.int32)
    n_fit = lib.oracle_refit_hits_f64(C.byref(g), C.c_float(float(geometry.bz_kgauss)), C.byref(prm._c()),
                                      C.c_uint32(len(row)), _ptr(sector), _ptr(row), _ptr(y), _ptr(z), _ptr(s),
                                      _ptr(ndf), _ptr(sec))
    return int(n_fit), s[0], s[1:6].copy(), s[6:21].copy(), s[21], int(ndf[0]), int(sec[0])


def canonical_tracks(track_task, track_hit_begin, track_nhits, hit_cluster):
    """Order of tracks by (task, first hit gid) - SPEC 7 / L4. Pure indexing."""
    first = hit_cluster[track_hit_begin.astype(np.int64)] if len(track_task) else np.zeros(0, np.uint32)
    return np.lexsort((first, track_task))
