"""Helpers of the -m gpu parity tests: run the CUDA path through the C ABI binding and
compare it with the CPU oracle on the same seeded inputs."""
from __future__ import annotations

import numpy as np

import oracle
from oracle import OracleParams


def oracle_params_for(batch, **over):
    return OracleParams(sigma_y=batch.sigma_y, sigma_z=batch.sigma_z, **over)


def tracker_params_for(batch, **over):
    from paper_1712_09434_b200 import TrackerParams
    return TrackerParams(sigma_y=batch.sigma_y, sigma_z=batch.sigma_z, **over)


def run_gpu(batch, debug=True, debug_tracklets=True, max_tracklets=0, counters=False, params_over=None,
            track_capacity=None, hit_capacity=None):
    """The whole path on cuda:0; returns the numpy dict of TrackResult.to_numpy()."""
    import torch
    from paper_1712_09434_b200 import Tracker
    dev = torch.device("cuda:0")
    trk = Tracker(batch.geometry, tracker_params_for(batch, **(params_over or {})))
    try:
        n = batch.n_clusters
        y = torch.from_numpy(np.ascontiguousarray(batch.y)).to(dev)
        z = torch.from_numpy(np.ascontiguousarray(batch.z)).to(dev)
        ro = torch.from_numpy(batch.row_offsets.astype(np.uint32).view(np.int32)).to(dev)
        n_dbg_trk = (n // 5 + 1) if debug_tracklets else 0
        out = trk.alloc_outputs(n, dev, debug=debug, debug_tracklets=n_dbg_trk, track_capacity=track_capacity,
                                hit_capacity=hit_capacity)
        ws = trk.alloc_workspace(trk.workspace_bytes(n, batch.n_tasks, max_tracklets), dev)
        trk.enable_counters(counters)
        trk.track_batch(y, z, ro, batch.n_tasks, out, ws, max_tracklets=max_tracklets)
        torch.cuda.synchronize()
        res = out.to_numpy()
        if counters:
            res["counters"] = trk.read_counters()
        return res
    finally:
        trk.close()


def run_oracle(batch, dump_tracklets=True, **over):
    return oracle.track(batch.geometry, batch.y, batch.z, batch.row_offsets, batch.n_tasks,
                        params=oracle_params_for(batch, **over), dump_tracklets=dump_tracklets)


def canonical(task, hit_begin, nhits, hits):
    first = hits[hit_begin.astype(np.int64)] if len(task) else np.zeros(0, np.int64)
    return np.lexsort((first.astype(np.int64), task.astype(np.int64)))


def compare(gpu, ref, n_rows, rtol=1e-4, check_tracklets=True):
    """Asserts the north_star bar: bit-exact links, start hits and hit lists; parameters within rtol.
    Returns a dict of the largest parameter deviations seen."""
    # a2, a3: links and cleaned links, gid-indexed, bit-exact
    for k, r in (("dbg_link_up", ref.link_up), ("dbg_link_dn", ref.link_dn), ("dbg_clean_up", ref.clean_up),
                 ("dbg_clean_dn", ref.clean_dn)):
        if k in gpu:
            np.testing.assert_array_equal(gpu[k][:len(r)], r, err_msg=k)
    # a4: start hits as a set
    if "dbg_start_hits" in gpu:
        ns = int(gpu["dbg_n_start_hits"][0])
        np.testing.assert_array_equal(np.sort(gpu["dbg_start_hits"][:ns].astype(np.int64)),
                                      ref.start_hits.astype(np.int64), err_msg="start hits")
    # a5: tracklets (before selection), matched by start-hit gid
    if check_tracklets and "dbg_tracklet_start" in gpu and ref.tracklet_start is not None:
        nk = gpu["n_tracklets"]
        assert nk == ref.n_tracklets, f"tracklets built: gpu {nk} oracle {ref.n_tracklets}"
        go = np.argsort(gpu["dbg_tracklet_start"][:nk].astype(np.int64), kind="stable")
        ro = np.argsort(ref.tracklet_start.astype(np.int64), kind="stable")
        np.testing.assert_array_equal(gpu["dbg_tracklet_start"][:nk][go].astype(np.int64),
                                      ref.tracklet_start[ro].astype(np.int64))
        np.testing.assert_array_equal(gpu["dbg_tracklet_nhits"][:nk][go].astype(np.int64),
                                      ref.tracklet_nhits[ro].astype(np.int64), err_msg="tracklet nHits")
        np.testing.assert_array_equal(gpu["dbg_tracklet_map"][:nk][go], ref.tracklet_map[ro],
                                      err_msg="tracklet row maps")
    # a6, a7: tracks
    assert gpu["status"] == 0, f"status bits {gpu['status']}"
    assert gpu["n_tracks"] == ref.n_tracks, f"tracks: gpu {gpu['n_tracks']} oracle {ref.n_tracks}"
    assert gpu["n_hits"] == len(ref.hit_cluster)
    go = canonical(gpu["track_task"], gpu["track_hit_begin"], gpu["track_nhits"], gpu["hit_cluster"])
    ro = canonical(ref.track_task, ref.track_hit_begin, ref.track_nhits, ref.hit_cluster)
    np.testing.assert_array_equal(gpu["track_task"][go].astype(np.int64), ref.track_task[ro].astype(np.int64))
    np.testing.assert_array_equal(gpu["track_nhits"][go].astype(np.int64), ref.track_nhits[ro].astype(np.int64))
    np.testing.assert_array_equal(gpu["track_ndf"][go], ref.track_ndf[ro])
    # hit lists, bit-exact, in ascending row order
    gh = np.concatenate([gpu["hit_cluster"][b:b + n] for b, n in
                         zip(gpu["track_hit_begin"][go].astype(np.int64), gpu["track_nhits"][go].astype(np.int64))]
                        or [np.zeros(0, np.int32)])
    rh = np.concatenate([ref.hit_cluster[b:b + n] for b, n in
                         zip(ref.track_hit_begin[ro].astype(np.int64), ref.track_nhits[ro].astype(np.int64))]
                        or [np.zeros(0, np.uint32)])
    np.testing.assert_array_equal(gh.astype(np.int64), rh.astype(np.int64), err_msg="per-track hit lists")
    assert len(np.unique(gh)) == len(gh), "a cluster is in two tracks"
    # fitted parameters and covariances: within rtol of the oracle (scale: the parameter's own sigma)
    dev = {}
    np.testing.assert_array_equal(gpu["track_x"][go], ref.track_x[ro])
    gp, rp = gpu["track_par"][:, go].astype(np.float64), ref.track_par[:, ro].astype(np.float64)
    gc, rc = gpu["track_cov"][:, go].astype(np.float64), ref.track_cov[:, ro].astype(np.float64)
    diag = [0, 2, 5, 9, 14]
    sig = np.sqrt(np.maximum(rc[diag], 0))
    scale_p = np.maximum(np.abs(rp), sig)
    dev["par_rel"] = float(np.max(np.abs(gp - rp) / np.maximum(scale_p, 1e-30))) if gp.size else 0.0
    k = 0
    scale_c = np.zeros_like(rc)
    for i in range(5):
        for j in range(i + 1):
            scale_c[k] = sig[i] * sig[j]
            k += 1
    scale_c = np.maximum(np.abs(rc), scale_c)
    dev["cov_rel"] = float(np.max(np.abs(gc - rc) / np.maximum(scale_c, 1e-30))) if gc.size else 0.0
    g2, r2 = gpu["track_chi2"][go].astype(np.float64), ref.track_chi2[ro].astype(np.float64)
    dev["chi2_rel"] = float(np.max(np.abs(g2 - r2) / np.maximum(np.abs(r2), 1.0))) if g2.size else 0.0
    dev["bit_exact"] = bool(np.array_equal(gpu["track_par"][:, go], ref.track_par[:, ro])
                            and np.array_equal(gpu["track_cov"][:, go], ref.track_cov[:, ro])
                            and np.array_equal(gpu["track_chi2"][go], ref.track_chi2[ro]))
    assert dev["par_rel"] <= rtol and dev["cov_rel"] <= rtol and dev["chi2_rel"] <= rtol, dev
    # north_star: "within 1e-4 relative".  Above, a parameter that is itself smaller than its own error is measured
    # against that error (a y of 1e-6 cm with sigma 0.03 cm has no meaningful relative deviation); wherever the value
    # exceeds its sigma the plain relative deviation must hold as well
    big = np.abs(rp) > sig
    dev["par_rel_plain"] = float(np.max(np.abs(gp - rp)[big] / np.abs(rp)[big])) if big.any() else 0.0
    assert dev["par_rel_plain"] <= rtol, dev
    return dev
