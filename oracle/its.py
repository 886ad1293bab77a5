"""ctypes wrapper of the ITS standalone tracker of the CPU oracle (oracle/tpc_oracle.cpp, SPEC 12) - TEST
INFRASTRUCTURE.  Marshals numpy arrays only."""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from .oracle import _load, _ptr


class _ItsGeom(C.Structure):
    _fields_ = [("R", C.c_float * 6), ("sig_rphi", C.c_float * 6), ("sig_z", C.c_float * 6), ("xx0", C.c_float * 6)]


_P_FLOATS = ("max_sinphi_pair", "max_dtan", "sig_sinphi", "sig_tan", "sig_vtx_xy", "sig_vtx_z", "chi2_max", "max_dx",
             "c0_sinphi", "c0_dzds", "c0_qpt", "turn_cov_scale", "max_sinphi")


class _ItsParams(C.Structure):
    _fields_ = [(n, C.c_float) for n in _P_FLOATS] + [("min_clusters", C.c_int32)]


class _ItsOut(C.Structure):
    _fields_ = [("capacity", C.c_uint32), ("event", C.c_void_p), ("cluster", C.c_void_p), ("n_clusters", C.c_void_p),
                ("frame", C.c_void_p), ("out_state", C.c_void_p), ("in_state", C.c_void_p), ("out_ndf", C.c_void_p),
                ("in_ndf", C.c_void_p), ("n_tracklets", C.c_uint32), ("n_tracks", C.c_uint32)]


@dataclass
class ItsParams:
    """Defaults of docs/ARITH_SPEC.md section 12 (the oracle's own copy)."""
    max_sinphi_pair: float = 0.03
    max_dtan: float = 0.02
    sig_sinphi: float = 0.002
    sig_tan: float = 0.004
    sig_vtx_xy: float = 0.01
    sig_vtx_z: float = 0.01
    chi2_max: float = 30.0
    max_dx: float = 2.0
    c0_sinphi: float = 1.0
    c0_dzds: float = 1.0
    c0_qpt: float = 100.0
    turn_cov_scale: float = 100.0
    max_sinphi: float = 0.95
    min_clusters: int = 4


@dataclass
class ItsResult:
    event: np.ndarray
    cluster: np.ndarray      # [n, 6] gid or -1
    n_clusters: np.ndarray
    frame: np.ndarray        # [n, 2] cos, sin of the tracklet's frame
    out_state: np.ndarray    # [n, 22] x, p[5], c[15], chi2 at the outermost attached cluster
    in_state: np.ndarray     # [n, 22] at the vertex plane
    out_ndf: np.ndarray
    in_ndf: np.ndarray
    n_tracklets: int


def its_track(geometry, x, y, z, layer_offsets, vertex, n_events: int, params: ItsParams | None = None,
              precision: str = "f32") -> ItsResult:
    lib = _load()
    lib.oracle_sizeof_its_out.restype = C.c_size_t
    assert lib.oracle_sizeof_its_out() == C.sizeof(_ItsOut)
    prm = params or ItsParams()
    dt = np.float32 if precision == "f32" else np.float64
    x, y, z = (np.ascontiguousarray(a, dtype=dt) for a in (x, y, z))
    lo = np.ascontiguousarray(layer_offsets, np.uint32)
    vt = np.ascontiguousarray(vertex, dtype=dt).reshape(-1)
    assert lo.shape[0] == n_events * 6 + 1 and vt.shape[0] == 3 * n_events
    g = _ItsGeom()
    for l in range(6):
        g.R[l], g.sig_rphi[l] = float(geometry.R[l]), float(geometry.sig_rphi[l])
        g.sig_z[l], g.xx0[l] = float(geometry.sig_z[l]), float(geometry.xx0[l])
    p = _ItsParams(**{n: getattr(prm, n) for n, _ in _ItsParams._fields_})
    cap = max(int(lo[-1]) // 2 + 1, 1)
    ev, ncl = np.empty(cap, np.uint32), np.empty(cap, np.uint32)
    cl = np.empty((cap, 6), np.int32)
    fr = np.empty((cap, 2), dt)
    so, si = np.empty((cap, 22), dt), np.empty((cap, 22), dt)
    no, ni = np.empty(cap, np.int32), np.empty(cap, np.int32)
    o = _ItsOut(cap, _ptr(ev), _ptr(cl), _ptr(ncl), _ptr(fr), _ptr(so), _ptr(si), _ptr(no), _ptr(ni), 0, 0)
    fn = lib.oracle_its_f32 if precision == "f32" else lib.oracle_its_f64
    fn.restype = C.c_int
    rc = fn(C.byref(g), C.c_float(float(geometry.bz_kgauss)), C.byref(p), C.c_uint32(n_events), _ptr(x), _ptr(y), _ptr(z),
            _ptr(lo), _ptr(vt), C.byref(o))
    if rc != 0:
        raise RuntimeError(f"oracle_its returned {rc}")
    n = o.n_tracks
    return ItsResult(ev[:n].copy(), cl[:n].copy(), ncl[:n].copy(), fr[:n].copy(), so[:n].copy(), si[:n].copy(),
                     no[:n].copy(), ni[:n].copy(), int(o.n_tracklets))
