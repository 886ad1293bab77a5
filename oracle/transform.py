"""CPU ORACLE of the TPC cluster transformation (docs/ARITH_SPEC.md section 10) - TEST INFRASTRUCTURE.

PAPER.md L77 (footnote 1): "The TPC cluster transformation map is needed to convert the raw TPC clusters from
TPC pad row, TPC pad, and time coordinates into x, y, and z coordinates taking into account the calibration";
L101, L213: the default or the fed-back calibration is applied, the cluster index does not change.

Plain numpy, one elementwise operation per SPEC step in the SPEC's order (numpy rounds every fp32 operation on
its own: no fused multiply-add), fp32 for parity and fp64 for the accuracy pins.  Shares nothing with
paper_1712_09434_b200/.  Pins: tests/test_oracle_transform.py (zero map = the nominal pad/time geometry and its
hand-computed values, round trip through the inverse nominal formula, a map that is a plane is reproduced
exactly, knots are reproduced at the knots, clamping outside the map, C-side mirror).
PARITY UNPINNED: the synthetic calibration's numbers (pad width, drift velocity, map size and amplitude).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class Calibration:
    """SPEC 10 calibration object (the oracle's own container)."""
    pad_pitch: np.ndarray   # float32 [n_rows]
    n_pads: np.ndarray      # int32 [n_rows]
    t0: float
    v_drift: float
    t_max: float
    corr: np.ndarray        # float32 [n_sectors, n_rows, MZ, MY, 2]  (dy, dz)


def transform(geometry, cal: Calibration, pad, time, row_offsets, n_tasks: int, precision: str = "f32"):
    """(pad, time) -> (y, z) for clusters sorted by (task,row); X1..X4."""
    R = np.float32 if precision == "f32" else np.float64
    pad = np.asarray(pad, R)
    time = np.asarray(time, R)
    ro = np.asarray(row_offsets, np.int64)
    nr, ns = int(geometry.n_rows), int(geometry.n_sectors)
    n = pad.shape[0]
    counts = np.diff(ro)
    tr = np.repeat(np.arange(n_tasks * nr), counts)
    row = tr % nr
    sec = (tr // nr) % ns
    a_side = 2 * sec < ns
    pitch = cal.pad_pitch.astype(R)[row]
    npad = cal.n_pads[row]
    z_max = R(geometry.z_max)
    # X1
    y0 = (pad - R(0.5) * (npad - 1).astype(R)) * pitch
    # X2
    zd = (time - R(cal.t0)) * R(cal.v_drift)
    z0 = np.where(a_side, z_max - zd, zd - z_max).astype(R)
    # X3
    MZ, MY = cal.corr.shape[2], cal.corr.shape[3]
    ky = (np.float32(MY - 1) / (cal.n_pads - 1).astype(np.float32)).astype(np.float32)   # host tables, fp32 divisions
    kz = np.float32(MZ - 1) / np.float32(cal.t_max)
    if precision != "f32":
        ky = (MY - 1) / (cal.n_pads - 1).astype(np.float64)
        kz = (MZ - 1) / float(cal.t_max)
    u = pad * ky.astype(R)[row]
    v = time * R(kz)
    u = np.fmin(np.fmax(u, R(0)), R(MY - 1))
    v = np.fmin(np.fmax(v, R(0)), R(MZ - 1))
    u = np.where(np.isnan(u), R(0), u)  # fmaxf(NaN, 0) = 0
    v = np.where(np.isnan(v), R(0), v)
    iu = np.minimum(u.astype(np.int64), MY - 2)
    iv = np.minimum(v.astype(np.int64), MZ - 2)
    fu = u - iu.astype(R)
    fv = v - iv.astype(R)
    m = cal.corr.astype(R)
    out = []
    for k in range(2):
        m00, m01 = m[sec, row, iv, iu, k], m[sec, row, iv, iu + 1, k]
        m10, m11 = m[sec, row, iv + 1, iu, k], m[sec, row, iv + 1, iu + 1, k]
        a = m00 + fu * (m01 - m00)
        b = m10 + fu * (m11 - m10)
        out.append(a + fv * (b - a))
    # X4
    y = y0 + out[0]
    z = z0 + out[1]
    assert y.shape[0] == n
    return y.astype(R), z.astype(R)
