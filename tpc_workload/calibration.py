"""Synthetic TPC read-out geometry and calibration map: seeded INPUT for the cluster transformation
(docs/ARITH_SPEC.md section 10).  Shared by the oracle's tests and the CUDA path's
tests and bench; it holds no part of the transformation itself - only the detector model that turns generated
(y, z) positions into the raw (pad, time) coordinates a TPC would have measured, and a smooth random correction
field sampled at the knots of the map.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class RawCalibration:
    pad_pitch: np.ndarray   # float32 [n_rows] cm
    n_pads: np.ndarray      # int32 [n_rows]
    t0: float               # time bin of a cluster at the end plate
    v_drift: float          # cm per time bin
    t_max: float            # time bin of the central electrode
    corr: np.ndarray        # float32 [n_sectors, n_rows, MZ, MY, 2] (dy, dz) in cm at the knots


def default_calibration(geometry, seed: int = 7, amplitude_cm: float = 0.3, my: int = 8, mz: int = 16,
                        zero_map: bool = False) -> RawCalibration:
    """Pads about 0.5 cm wide, 1000 time bins of drift, corrections of a few millimetres that vary smoothly
    over a row (a handful of random harmonics per sector)."""
    X = geometry.row_x.astype(np.float64)
    half = X * float(geometry.tan_half_angle)
    n_pads = (2 * np.floor(half / 0.5)).astype(np.int32)
    pitch = (2.0 * half / n_pads).astype(np.float32)
    t_max = 1000.0
    v = float(geometry.z_max) / t_max
    ns, nr = int(geometry.n_sectors), int(geometry.n_rows)
    corr = np.zeros((ns, nr, mz, my, 2), np.float32)
    if not zero_map:
        rng = np.random.Generator(np.random.PCG64(seed))
        uu = np.linspace(0.0, 1.0, my)[None, None, None, :]
        vv = np.linspace(0.0, 1.0, mz)[None, None, :, None]
        rr = np.linspace(0.0, 1.0, nr)[None, :, None, None]
        for k in range(2):
            f = np.zeros((ns, nr, mz, my))
            for _ in range(4):
                ph = rng.uniform(0, 2 * np.pi, (ns, 1, 1, 1))
                wu, wv, wr = rng.uniform(0.5, 2.5, 3)
                f += rng.uniform(0.3, 1.0) * np.sin(2 * np.pi * (wu * uu + wv * vv + wr * rr) + ph)
            corr[..., k] = (amplitude_cm / 2.0 * f).astype(np.float32)
    return RawCalibration(pad_pitch=pitch, n_pads=n_pads, t0=0.0, v_drift=v, t_max=t_max, corr=corr)


def raw_from_yz(geometry, cal: RawCalibration, y, z, row_offsets, n_tasks: int):
    """The (pad, time) a cluster at local (y, z) is read out at, by the NOMINAL geometry (fp64, then fp32)."""
    nr, ns = int(geometry.n_rows), int(geometry.n_sectors)
    counts = np.diff(np.asarray(row_offsets, np.int64))
    tr = np.repeat(np.arange(n_tasks * nr), counts)
    row, sec = tr % nr, (tr // nr) % ns
    a_side = 2 * sec < ns
    y = np.asarray(y, np.float64)
    z = np.asarray(z, np.float64)
    pad = y / cal.pad_pitch.astype(np.float64)[row] + 0.5 * (cal.n_pads[row] - 1)
    zd = np.where(a_side, float(geometry.z_max) - z, z + float(geometry.z_max))
    time = cal.t0 + zd / cal.v_drift
    return pad.astype(np.float32), time.astype(np.float32)
