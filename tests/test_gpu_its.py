"""-m gpu parity of the ITS standalone tracker (SPEC 12, tpc_its_track_batch) against the CPU oracle: the same tracks
in the same order, cluster for cluster; frames, outward and inward states within 1e-4 (reported bit-identical)."""
from __future__ import annotations

import numpy as np
import pytest

from oracle.its import its_track, ItsParams
from tpc_workload import default_its_geometry, generate_its_events

pytestmark = pytest.mark.gpu


def run_gpu(b, geom, params=None):
    import torch
    from paper_1712_09434_b200 import ItsTracker
    dev = torch.device("cuda:0")
    trk = ItsTracker(geom, params)
    try:
        t = lambda a, dt=None: torch.from_numpy(np.ascontiguousarray(a if dt is None else a.astype(dt))).to(dev)  # noqa: E731
        out = trk.track_batch(t(b.x), t(b.y), t(b.z), t(b.layer_offsets.astype(np.uint32).view(np.int32)),
                              t(b.vertex.astype(np.float32).reshape(-1)), b.n_events)
        torch.cuda.synchronize()
        h = out["header"].cpu().numpy()
        n = int(h[0])
        res = {k: v[:n].cpu().numpy() for k, v in out.items() if k not in ("header", "_workspace")}
        res["header"] = h
        return res
    finally:
        trk.close()


def compare(g, r, rtol=1e-4):
    assert g["header"][2] == 0 and g["header"][0] == len(r.event) and g["header"][1] == r.n_tracklets
    np.testing.assert_array_equal(g["event"], r.event.astype(np.int32))
    np.testing.assert_array_equal(g["cluster"], r.cluster)
    np.testing.assert_array_equal(g["n_clusters"], r.n_clusters.astype(np.int32))
    np.testing.assert_array_equal(g["out_ndf"], r.out_ndf)
    np.testing.assert_array_equal(g["in_ndf"], r.in_ndf)
    exact = True
    for k, ref in (("frame", r.frame), ("out_state", r.out_state), ("in_state", r.in_state)):
        a, b_ = g[k].astype(np.float64), ref.astype(np.float64)
        if k == "frame":
            assert np.max(np.abs(a - b_)) <= rtol
        else:
            sig = np.sqrt(np.maximum(b_[:, 6:21][:, [0, 2, 5, 9, 14]], 0))
            scale = np.maximum(np.abs(b_[:, 1:6]), sig)
            assert np.max(np.abs(a[:, 1:6] - b_[:, 1:6]) / np.maximum(scale, 1e-30)) <= rtol, k
            assert np.max(np.abs(a[:, 0] - b_[:, 0])) <= rtol * 50.0
        exact &= bool(np.array_equal(g[k], ref))
    return exact


@pytest.mark.parametrize("n_events,n_tracks,seed", [(1, 50, 1), (4, 400, 2), (16, 1500, 3)])
def test_its_tracker_matches_the_oracle(n_events, n_tracks, seed):
    geom = default_its_geometry()
    b = generate_its_events(geom, n_events, n_tracks, seed=seed, pt_range=(0.15, 5.0), noise_frac=0.1)
    r = its_track(geom, b.x, b.y, b.z, b.layer_offsets, b.vertex, b.n_events)
    g = run_gpu(b, geom)
    exact = compare(g, r)
    assert len(r.event) > 0.9 * n_events * n_tracks * 0.8
    print(f"ITS {n_events} events x {n_tracks} tracks: {b.n_clusters} clusters, {r.n_tracklets} tracklets, "
          f"{len(r.event)} tracks; bit-identical states: {exact}")


def test_its_parameters_bz0_and_empty():
    geom = default_its_geometry(xx0=0.0)
    b = generate_its_events(geom, 3, 200, seed=7, noise_frac=0.3)
    for over in (dict(chi2_max=5.0), dict(min_clusters=6), dict(max_sinphi_pair=0.01, max_dtan=0.005),
                 dict(sig_vtx_xy=0.1, sig_vtx_z=1.0), dict(turn_cov_scale=1.0)):
        r = its_track(geom, b.x, b.y, b.z, b.layer_offsets, b.vertex, b.n_events, params=ItsParams(**over))
        compare(run_gpu(b, geom, over), r)
    import dataclasses
    g0 = dataclasses.replace(geom, bz_kgauss=0.0)
    b0 = generate_its_events(dataclasses.replace(geom, bz_kgauss=1e-6), 2, 100, seed=8, pt_range=(50.0, 100.0))
    compare(run_gpu(b0, g0), its_track(g0, b0.x, b0.y, b0.z, b0.layer_offsets, b0.vertex, b0.n_events))
    empty = dataclasses.replace(b, x=b.x[:0], y=b.y[:0], z=b.z[:0], layer_offsets=np.zeros(19, np.uint32))
    ge = run_gpu(empty, geom)
    assert ge["header"][0] == 0 and ge["header"][1] == 0
