"""Pins of SPEC 10 (cluster transformation: pad row, pad, time -> x, y, z with a calibration map; PAPER.md L77,
L101, L213) on the CPU oracle (oracle/transform.py).  Expectations are hand-computed or closed forms, never the
oracle's own expressions re-typed."""
from __future__ import annotations

import numpy as np

from oracle.transform import Calibration, transform
from tpc_workload import default_geometry, generate_config, default_calibration, raw_from_yz

GEOM = default_geometry()


def cal_of(raw) -> Calibration:
    return Calibration(raw.pad_pitch, raw.n_pads, raw.t0, raw.v_drift, raw.t_max, raw.corr)


def one_cluster_batch(task, row, geom=GEOM):
    ro = np.zeros(geom.n_sectors * geom.n_rows + 1, np.uint32)
    ro[task * geom.n_rows + row + 1:] = 1
    return ro


def test_nominal_geometry_hand_computed():
    """X1, X2 with a zero map: a row of 100 pads of 0.625 cm, 1000 time bins over 250 cm."""
    raw = default_calibration(GEOM, zero_map=True)
    raw.n_pads[:] = 100
    raw.pad_pitch[:] = 0.625   # a binary fraction: exact in the fp32 table
    raw.t0, raw.v_drift, raw.t_max = 10.0, 0.25, 1010.0
    cal = cal_of(raw)
    # pad 49.5 is the centre of the row; pad 0 is 49.5 pads to the left; time 10 is the end plate (z = 250)
    for (pad, time, y_want, z_want) in ((49.5, 10.0, 0.0, 250.0), (0.0, 10.0, -30.9375, 250.0),
                                        (99.0, 410.0, 30.9375, 150.0), (59.5, 1010.0, 6.25, 0.0)):
        y, z = transform(GEOM, cal, [pad], [time], one_cluster_batch(3, 40), GEOM.n_sectors, precision="f64")
        assert abs(y[0] - y_want) < 1e-6 and abs(z[0] - z_want) < 1e-6 
        yc, zc = transform(GEOM, cal, [pad], [time], one_cluster_batch(3 + 18, 40), GEOM.n_sectors, precision="f64")
        assert abs(yc[0] - y_want) < 1e-6 and abs(zc[0] + z_want) < 1e-6  # C side: z mirrored, y not


def test_zero_map_inverts_the_readout_model():
    """(y, z) -> (pad, time) by the detector model of the generator -> transform gives (y, z) back: fp32 inputs carry
    half an ulp of a 1000-bin time (3e-5 bins = 8e-6 cm), fp64 is exact to 1e-9 on fp64 raw coordinates."""
    b = generate_config(1)
    raw = default_calibration(b.geometry, zero_map=True)
    pad, time = raw_from_yz(b.geometry, raw, b.y, b.z, b.row_offsets, b.n_tasks)
    y, z = transform(b.geometry, cal_of(raw), pad, time, b.row_offsets, b.n_tasks, precision="f32")
    assert np.max(np.abs(y - b.y)) < 2e-5 and np.max(np.abs(z - b.z)) < 1e-4
    assert y.dtype == np.float32 and len(y) == b.n_clusters          # L213: same index, same count


def test_a_plane_is_interpolated_exactly_and_knots_are_reproduced():
    """X3: bilinear interpolation reproduces any map of the form c0 + c1*u + c2*v (u, v = knot coordinates), and
    returns the knot value at a knot, whatever the neighbours are."""
    rng = np.random.default_rng(1)
    raw = default_calibration(GEOM, zero_map=True)
    MZ, MY = raw.corr.shape[2], raw.corr.shape[3]
    iu, iv = np.meshgrid(np.arange(MY), np.arange(MZ))
    raw.corr[..., 0] = (0.1 + 0.02 * iu - 0.03 * iv).astype(np.float32)
    raw.corr[..., 1] = (-0.2 + 0.05 * iu + 0.01 * iv).astype(np.float32)
    cal = cal_of(raw)
    row, task = 77, 5
    npad = int(raw.n_pads[row])
    for _ in range(50):
        pad, time = rng.uniform(0, npad - 1), rng.uniform(0, raw.t_max)
        u, v = pad * (MY - 1) / (npad - 1), time * (MZ - 1) / raw.t_max
        y, z = transform(GEOM, cal, [pad], [time], one_cluster_batch(task, row), GEOM.n_sectors, precision="f64")
        y_nom = (pad - 0.5 * (npad - 1)) * float(raw.pad_pitch[row])
        z_nom = GEOM.z_max - time * raw.v_drift
        assert abs((y[0] - y_nom) - (0.1 + 0.02 * u - 0.03 * v)) < 1e-7
        assert abs((z[0] - z_nom) - (-0.2 + 0.05 * u + 0.01 * v)) < 1e-7
    raw2 = default_calibration(GEOM, seed=3)
    cal2 = cal_of(raw2)
    for (ku, kv) in ((0, 0), (3, 5), (MY - 1, MZ - 1), (MY - 1, 0), (2, MZ - 1)):
        pad, time = ku * (npad - 1) / (MY - 1), kv * raw2.t_max / (MZ - 1)
        y, z = transform(GEOM, cal2, [pad], [time], one_cluster_batch(task, row), GEOM.n_sectors, precision="f64")
        y_nom = (pad - 0.5 * (npad - 1)) * float(raw2.pad_pitch[row])
        z_nom = GEOM.z_max - time * raw2.v_drift
        assert abs((y[0] - y_nom) - float(raw2.corr[task, row, kv, ku, 0])) < 1e-6
        assert abs((z[0] - z_nom) - float(raw2.corr[task, row, kv, ku, 1])) < 1e-6


def test_map_is_per_sector_and_row_and_clamped_outside():
    raw = default_calibration(GEOM, zero_map=True)
    raw.corr[4, 10, :, :, 0] = 0.25          # only sector 4, row 10 is corrected
    raw.corr[4, 10, :, :, 1] = -0.5
    cal = cal_of(raw)
    npad = int(raw.n_pads[10])
    for task, row, dy, dz in ((4, 10, 0.25, -0.5), (4, 11, 0.0, 0.0), (5, 10, 0.0, 0.0), (4 + 36, 10, 0.25, -0.5)):
        ro = np.zeros(2 * GEOM.n_sectors * GEOM.n_rows + 1, np.uint32)
        ro[task * GEOM.n_rows + row + 1:] = 1
        y, z = transform(GEOM, cal, [10.0], [100.0], ro, 2 * GEOM.n_sectors, precision="f64")
        assert abs(y[0] - ((10.0 - 0.5 * (int(raw.n_pads[row]) - 1)) * float(raw.pad_pitch[row]) + dy)) < 1e-9
        assert abs(z[0] - (GEOM.z_max - 100.0 * raw.v_drift + dz)) < 1e-9
    # beyond the last knot the edge value is used (clamp), also for NaN-free garbage like negative pads
    raw.corr[4, 10, :, -1, 0] = 1.0
    y, _ = transform(GEOM, cal_of(raw), [npad + 5.0], [100.0], one_cluster_batch(4, 10), GEOM.n_sectors, precision="f64")
    assert abs(y[0] - ((npad + 5.0 - 0.5 * (npad - 1)) * float(raw.pad_pitch[10]) + 1.0)) < 1e-9


def test_f32_follows_f64():
    b = generate_config(0)
    raw = default_calibration(b.geometry, seed=5)
    pad, time = raw_from_yz(b.geometry, raw, b.y, b.z, b.row_offsets, b.n_tasks)
    y32, z32 = transform(b.geometry, cal_of(raw), pad, time, b.row_offsets, b.n_tasks, precision="f32")
    y64, z64 = transform(b.geometry, cal_of(raw), pad, time, b.row_offsets, b.n_tasks, precision="f64")
    assert np.max(np.abs(y32 - y64)) < 2e-5 and np.max(np.abs(z32 - z64)) < 1e-4
    assert 0.05 < np.max(np.abs(y32 - b.y)) < 0.6   # the map moves clusters by millimetres
