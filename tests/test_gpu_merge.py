"""-m gpu parity of the sector-segment merger + refit (SPEC 9, include/tpc_tracker.h tpc_merge_refit) against
the CPU oracle on the same seeded inputs: links bit-exact (as pairs of first-hit gids: track order is free, L4),
chains and hit counts bit-exact, refitted parameters within 1e-4 (reported bit-identical)."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import gpu_helpers as G
from tpc_workload import generate_config

pytestmark = pytest.mark.gpu


def run_gpu_merge(batch, chi2_max=None, max_row_gap=None, params_over=None, n_slices=1):
    import torch
    from paper_1712_09434_b200 import Tracker
    dev = torch.device("cuda:0")
    trk = Tracker(batch.geometry, G.tracker_params_for(batch, **(params_over or {})))
    try:
        n = batch.n_clusters
        y = torch.from_numpy(np.ascontiguousarray(batch.y)).to(dev)
        z = torch.from_numpy(np.ascontiguousarray(batch.z)).to(dev)
        ro = torch.from_numpy(batch.row_offsets.astype(np.uint32).view(np.int32)).to(dev)
        out = trk.alloc_outputs(n, dev)
        ws = trk.alloc_workspace(trk.workspace_bytes(n, batch.n_tasks), dev)
        tcap = int(out.track_task.shape[0])
        merged = trk.alloc_merged(tcap, dev)
        mws = trk.alloc_workspace(trk.merge_workspace_bytes(tcap, batch.n_tasks), dev)
        trk.track_batch(y, z, ro, batch.n_tasks, out, ws)
        trk.merge_refit(y, z, ro, batch.n_tasks, out, merged, ws, mws, chi2_max=chi2_max, max_row_gap=max_row_gap,
                        n_slices=n_slices)
        torch.cuda.synchronize()
        g = out.to_numpy()
        g.update(merged.to_numpy(g["n_tracks"]))
        return g
    finally:
        trk.close()


def compare_merge(g, ref, mref, rtol=1e-4):
    assert g["status"] == 0 and g["n_tracks"] == ref.n_tracks
    fg = g["hit_cluster"][g["track_hit_begin"].astype(np.int64)].astype(np.int64)
    fr = ref.hit_cluster[ref.track_hit_begin.astype(np.int64)].astype(np.int64)
    links_g = {(int(fg[i]), int(fg[g["seg_next"][i]])) for i in np.nonzero(g["seg_next"] >= 0)[0]}
    links_r = {(int(fr[i]), int(fr[mref.next[i]])) for i in np.nonzero(mref.next >= 0)[0]}
    assert links_g == links_r, f"links differ: gpu {len(links_g)} oracle {len(links_r)}"
    assert g["n_links"] == mref.n_links == len(links_r)
    for i in np.nonzero(g["seg_next"] >= 0)[0]:
        assert g["seg_prev"][g["seg_next"][i]] == i
    assert g["n_merged"] == len(mref.merged_first)
    # merged tracks matched by the first-hit gid of their innermost segment
    by = {int(fr[f]): k for k, f in enumerate(mref.merged_first)}
    order = np.array([by[int(fg[f])] for f in g["merged_first"]], np.int64)
    assert len(set(order.tolist())) == len(order)
    assert np.all(np.diff(g["merged_first"].astype(np.int64)) > 0), "merged tracks are in the order of their first segment"
    for f in ("merged_nseg", "merged_nhits", "merged_nfit", "merged_sector", "merged_ndf"):
        np.testing.assert_array_equal(g[f].astype(np.int64), getattr(mref, f)[order].astype(np.int64), err_msg=f)
    np.testing.assert_array_equal(g["merged_x"], mref.merged_x[order])
    gp, rp = g["merged_par"].astype(np.float64), mref.merged_par[:, order].astype(np.float64)
    gc, rc = g["merged_cov"].astype(np.float64), mref.merged_cov[:, order].astype(np.float64)
    sig = np.sqrt(np.maximum(rc[[0, 2, 5, 9, 14]], 0))
    dev_p = float(np.max(np.abs(gp - rp) / np.maximum(np.maximum(np.abs(rp), sig), 1e-30))) if gp.size else 0.0
    assert dev_p <= rtol, f"refit parameters deviate by {dev_p:.2e}"
    k, scale = 0, np.zeros_like(rc)
    for i in range(5):
        for j in range(i + 1):
            scale[k] = sig[i] * sig[j]
            k += 1
    dev_c = float(np.max(np.abs(gc - rc) / np.maximum(np.maximum(np.abs(rc), scale), 1e-30))) if gc.size else 0.0
    assert dev_c <= rtol, f"refit covariances deviate by {dev_c:.2e}"
    g2, r2 = g["merged_chi2"].astype(np.float64), mref.merged_chi2[order].astype(np.float64)
    assert np.all(np.abs(g2 - r2) <= rtol * np.maximum(np.abs(r2), 1.0))
    return dict(par_rel=dev_p, cov_rel=dev_c, bit_exact=bool(np.array_equal(g["merged_par"], mref.merged_par[:, order])
                                                              and np.array_equal(g["merged_cov"], mref.merged_cov[:, order])))


@pytest.mark.parametrize("cfg", [1, 2])
def test_merge_refit_matches_the_oracle(cfg):
    b = generate_config(cfg)
    g = run_gpu_merge(b)
    prm = G.oracle_params_for(b)
    ref = oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, params=prm)
    mref = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, ref, params=prm)
    dev = compare_merge(g, ref, mref)
    assert mref.n_links > 100
    print(f"config {cfg}: {ref.n_tracks} sector tracks, {mref.n_links} links, {len(mref.merged_first)} merged; {dev}")


def test_merge_refit_multi_event_batch_and_cuts():
    """Four events in one call (links never cross events), and the two cuts away from their defaults."""
    b = generate_config(3, n_events=4)
    prm = G.oracle_params_for(b)
    ref = oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, params=prm)
    for chi2_max, gap in ((50.0, 8), (5.0, 8), (50.0, 1), (1e6, 20)):
        g = run_gpu_merge(b, chi2_max=chi2_max, max_row_gap=gap)
        mref = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, ref, params=prm, chi2_max=chi2_max,
                                  max_row_gap=gap)
        compare_merge(g, ref, mref)
    ns = b.geometry.n_sectors
    i = np.nonzero(g["seg_next"] >= 0)[0]
    assert np.all(g["track_task"][i] // ns == g["track_task"][g["seg_next"][i]] // ns)


def test_merge_refit_single_sector_and_empty():
    """Config 0 has one sector (no neighbours): no links, every track refitted alone; an empty batch gives nothing."""
    b = generate_config(0)
    g = run_gpu_merge(b)
    prm = G.oracle_params_for(b)
    ref = oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, params=prm)
    mref = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, ref, params=prm)
    assert mref.n_links == 0
    compare_merge(g, ref, mref)
    from tpc_workload import take_tasks
    e, _ = take_tasks(generate_config(1), [])   # every task empty
    ge = run_gpu_merge(e)
    assert ge["n_tracks"] == 0 and ge["n_merged"] == 0 and ge["n_links"] == 0


def test_time_frame_mode_matches_the_oracle():
    """SPEC 11: six overlapping peripheral events in one frame of four slices (144 slice-sector tasks), tracker with
    nf_z_projection = 0, merger across sectors AND slices: tracks, links and refit identical to the oracle's; and a
    second frame in the same call (frames never mix)."""
    from tpc_workload import default_geometry, generate_event, make_frame, concat_batches, CONFIGS
    geom = default_geometry()
    spec = CONFIGS[1]["spec"]
    frames = []
    for f in range(2):
        evs = [generate_event(geom, spec, 400 + 10 * f + i) for i in range(6)]
        shifts = np.sort(np.random.default_rng(5 + f).uniform(0, 750, 6))
        frames.append(make_frame(evs, shifts, 250.0, 4, seed=9 + f))
    b = concat_batches(frames)
    over = dict(nf_z_projection=0, nf_hz=2.5)
    prm = G.oracle_params_for(b, **over)
    ref = oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, params=prm)
    mref = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, ref, params=prm, n_slices=4)
    g = run_gpu_merge(b, params_over=over, n_slices=4)
    G.compare(g, ref, b.geometry.n_rows, check_tracklets=False)
    dev = compare_merge(g, ref, mref)
    ns = geom.n_sectors
    i = np.nonzero(g["seg_next"] >= 0)[0]
    ti, tj = g["track_task"][i].astype(np.int64), g["track_task"][g["seg_next"][i]].astype(np.int64)
    assert np.all(ti // (4 * ns) == tj // (4 * ns))           # same frame
    assert np.sum(ti // ns != tj // ns) > 300                 # links across slices exist
    print(f"frames: {ref.n_tracks} tracks, {mref.n_links} links, {len(mref.merged_first)} merged; {dev}")


def test_frame_slicer_matches_the_oracle_and_feeds_the_tracker():
    """SLICE: a frame given unsliced (sorted by (sector,row)) is sliced on the device exactly as oracle/frames.py does
    (arrays, source indices, row offsets identical); tracker + merger on the device's slices equal the oracle's on
    the oracle's slices; the source indices give the clusters of a track back in the unsliced numbering."""
    import torch
    from oracle.frames import slice_frames as oracle_slice
    from paper_1712_09434_b200 import slice_frames, Tracker
    from tpc_workload import default_geometry, generate_event, make_frame, CONFIGS
    import dataclasses
    geom = default_geometry()
    evs = [generate_event(geom, CONFIGS[1]["spec"], 600 + i) for i in range(5)]
    whole = make_frame(evs, [0.0, 130.0, 377.0, 512.0, 740.0], 1000.0, 1, seed=2)   # one slice = not yet sliced
    ns, nr, n_sl = geom.n_sectors, geom.n_rows, 4
    yo, zo, so, roo = oracle_slice(whole.y, whole.z, whole.row_offsets, ns, ns, nr, 250.0, n_sl)
    dev = torch.device("cuda:0")
    y = torch.from_numpy(whole.y).to(dev); z = torch.from_numpy(whole.z).to(dev)
    ro = torch.from_numpy(whole.row_offsets.astype(np.uint32).view(np.int32)).to(dev)
    yg, zg, sg, rog = slice_frames(y, z, ro, ns, ns, nr, 250.0, n_sl)
    torch.cuda.synchronize()
    assert np.array_equal(yg.cpu().numpy(), yo) and np.array_equal(zg.cpu().numpy(), zo)
    assert np.array_equal(sg.cpu().numpy().view(np.uint32), so)
    assert np.array_equal(rog.cpu().numpy().view(np.uint32), roo)
    sliced = dataclasses.replace(whole, y=yo, z=zo, row_offsets=roo, n_tasks=ns * n_sl, x=whole.x[so],
                                 charge=whole.charge[so], truth_track=whole.truth_track[so],
                                 truth_leg=whole.truth_leg[so], truth_state=whole.truth_state[so])
    over = dict(nf_z_projection=0, nf_hz=2.5)
    prm = G.oracle_params_for(sliced, **over)
    ref = oracle.track(sliced.geometry, yo, zo, roo, ns * n_sl, params=prm)
    mref = oracle.merge_refit(sliced.geometry, yo, zo, roo, ns * n_sl, ref, params=prm, n_slices=n_sl)
    trk = Tracker(sliced.geometry, G.tracker_params_for(sliced, **over))
    try:
        n = whole.n_clusters
        out = trk.alloc_outputs(n, dev)
        ws = trk.alloc_workspace(trk.workspace_bytes(n, ns * n_sl), dev)
        tcap = int(out.track_task.shape[0])
        merged = trk.alloc_merged(tcap, dev)
        mws = trk.alloc_workspace(trk.merge_workspace_bytes(tcap, ns * n_sl), dev)
        trk.track_batch(yg, zg, rog, ns * n_sl, out, ws)
        trk.merge_refit(yg, zg, rog, ns * n_sl, out, merged, ws, mws, n_slices=n_sl)
        torch.cuda.synchronize()
        g = out.to_numpy()
        g.update(merged.to_numpy(g["n_tracks"]))
    finally:
        trk.close()
    G.compare(g, ref, nr, check_tracklets=False)
    compare_merge(g, ref, mref)
    orig = so[g["hit_cluster"].astype(np.int64)]                      # hits in the numbering of the unsliced frame
    assert np.array_equal(whole.y[orig], yo[g["hit_cluster"].astype(np.int64)])
    empty = slice_frames(y[:0], z[:0], torch.zeros(ns * nr + 1, dtype=torch.int32, device=dev), ns, ns, nr, 250.0, n_sl)
    torch.cuda.synchronize()
    assert empty[0].numel() == 0 and int(empty[3].abs().sum()) == 0
