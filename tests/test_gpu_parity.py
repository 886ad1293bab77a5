"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle on the same seeded
inputs.  Bar (BASELINE.json north_star): bit-exact neighbour links, cleaned links, start hits,
tracklet row maps and per-track cluster index lists; fitted parameters, covariances and chi2 within
RTOL = 1e-4 relative (both sides run the same non-contracted fp32 sequence of docs/ARITH_SPEC.md,
so they are in fact expected to be bit-identical, which is reported but not required).
"""
from __future__ import annotations

import numpy as np
import pytest

from tpc_workload import generate_config, take_tasks, concat_batches, default_geometry
from helpers import batch_from_rows
import gpu_helpers as G

pytestmark = pytest.mark.gpu
RTOL = 1e-4  # north_star: "fitted track parameters and covariances must agree within 1e-4 relative"


@pytest.fixture(scope="module")
def cfg2():
    return generate_config(2)


# ---- element by element, whole configs ------------------------------------------------------
@pytest.mark.parametrize("config", [0, 1])
def test_small_configs_every_stage(config):
    b = generate_config(config)
    gpu = G.run_gpu(b)
    ref = G.run_oracle(b)
    dev = G.compare(gpu, ref, b.geometry.n_rows, rtol=RTOL)
    assert ref.n_tracks > 0
    print(f"config {config}: {b.n_clusters} clusters, {ref.n_tracks} tracks, deviations {dev}")


def test_config2_central_event_every_stage(cfg2):
    """One central event: 2.5 M clusters, 5 700 row blocks of 28..570 clusters (several tiles + ragged tails)."""
    gpu = G.run_gpu(cfg2)
    ref = G.run_oracle(cfg2)
    dev = G.compare(gpu, ref, cfg2.geometry.n_rows, rtol=RTOL)
    print(f"config 2: {cfg2.n_clusters} clusters, {ref.n_tracks} tracks, deviations {dev}")


def test_config4_stress_every_stage():
    """50 000 tracks, 20 % noise, wider errors: long candidate lists in both searches."""
    b = generate_config(4)
    gpu = G.run_gpu(b)
    ref = G.run_oracle(b)
    dev = G.compare(gpu, ref, b.geometry.n_rows, rtol=RTOL)
    print(f"config 4: {b.n_clusters} clusters, {ref.n_tracks} tracks, deviations {dev}")


# ---- the bench launch configuration at full size, EVERY task against the oracle ----------------
_POOL_B = None


def _oracle_task(task):
    """Worker of the process pool: the oracle on one sector task; tracks as {hit gids (batch numbering): record}."""
    sub, sel = take_tasks(_POOL_B, [task])
    ref = G.run_oracle(sub, dump_tracklets=False)
    out = {}
    for t in range(ref.n_tracks):
        key = tuple(sel[ref.track_hits(t).astype(np.int64)].tolist())
        out[key] = (int(ref.track_ndf[t]), float(ref.track_x[t]), ref.track_par[:, t].copy(), ref.track_cov[:, t].copy(),
                    float(ref.track_chi2[t]))
    return task, out


def test_config3_full_batch_all_576_tasks():
    """Config 3 exactly as bench.py runs it (16 events, 576 tasks, one call, no debug outputs, default
    capacities).  Tasks are independent, so the oracle computes them one by one (a process
    pool over the host cores; about one core-minute) and EVERY track of EVERY task must match: hit lists
    bit-exact, ndf and x equal, parameters / covariances / chi2 within RTOL."""
    global _POOL_B
    import multiprocessing as mp
    import os
    b = generate_config(3, workers=8)
    gpu = G.run_gpu(b, debug=False, debug_tracklets=False)
    assert gpu["status"] == 0
    nr = b.geometry.n_rows
    hits = gpu["hit_cluster"].astype(np.int64)
    assert len(np.unique(hits)) == len(hits)
    assert gpu["n_hits"] == len(hits) and int(gpu["track_nhits"].sum()) == len(hits)
    assert int(gpu["track_nhits"].min()) >= 10
    tr_of = np.searchsorted(b.row_offsets.astype(np.int64), hits, side="right") - 1
    beg = gpu["track_hit_begin"].astype(np.int64)
    seg = np.repeat(np.arange(len(beg)), gpu["track_nhits"].astype(np.int64))
    assert np.array_equal(tr_of // nr, gpu["track_task"].astype(np.int64)[seg]), "a hit outside its track's task"
    same = seg[1:] == seg[:-1]
    assert np.all((tr_of[1:] > tr_of[:-1])[same]), "hits not in ascending row order"
    got = {}
    for t in range(gpu["n_tracks"]):
        got[tuple(hits[beg[t]:beg[t] + int(gpu["track_nhits"][t])].tolist())] = t
    assert len(got) == gpu["n_tracks"]
    G.run_oracle(take_tasks(b, [0])[0], dump_tracklets=False)  # builds / loads the oracle before the fork
    _POOL_B = b
    with mp.get_context("fork").Pool(min(len(os.sched_getaffinity(0)), 64)) as pool:
        results = pool.map(_oracle_task, range(b.n_tasks), chunksize=4)
    _POOL_B = None
    n_ref = 0
    worst = 0.0
    for task, ref in results:
        n_ref += len(ref)
        for key, (ndf, x, rp, rc, chi2) in ref.items():
            assert key in got, f"task {task}: an oracle track is missing on the GPU"
            g = got[key]
            assert int(gpu["track_task"][g]) == task and int(gpu["track_ndf"][g]) == ndf
            assert float(gpu["track_x"][g]) == x
            rp, gp = rp.astype(np.float64), gpu["track_par"][:, g].astype(np.float64)
            rc, gc = rc.astype(np.float64), gpu["track_cov"][:, g].astype(np.float64)
            sig = np.sqrt(np.maximum(rc[[0, 2, 5, 9, 14]], 0))
            sc = np.array([sig[i] * sig[j] for i in range(5) for j in range(i + 1)])
            dp = np.max(np.abs(gp - rp) / np.maximum(np.maximum(np.abs(rp), sig), 1e-30))
            dc = np.max(np.abs(gc - rc) / np.maximum(np.maximum(np.abs(rc), sc), 1e-30))
            worst = max(worst, dp, dc, abs(float(gpu["track_chi2"][g]) - chi2) / max(abs(chi2), 1.0))
    assert n_ref == gpu["n_tracks"], f"tracks: gpu {gpu['n_tracks']} oracle {n_ref}"
    assert worst <= RTOL, worst
    print(f"config 3: {b.n_clusters} clusters, {b.n_tasks} tasks, {n_ref} tracks identical; worst deviation {worst:.2e}")


# ---- every parameter of tpc_params, away from its default ----------------------------------------
@pytest.mark.parametrize("over", [
    dict(max_row_gap=0), dict(max_row_gap=1), dict(min_seed_hits=3), dict(min_seed_hits=8),
    dict(min_track_hits=5), dict(min_track_hits=30), dict(accept_k2=4.0), dict(search_max=0.5),
    dict(turn_cov_scale=1.0), dict(max_sinphi=0.5), dict(nf_hy=1.0, nf_hz=3.0, nf_chi2_max=20.0),
    dict(c0_sinphi=0.1, c0_dzds=0.1, c0_qpt=10.0),
])
def test_parameter_sweep_config1(over):
    b = generate_config(1)
    gpu = G.run_gpu(b, params_over=over)
    ref = G.run_oracle(b, **over)
    G.compare(gpu, ref, b.geometry.n_rows, rtol=RTOL)
    assert ref.n_tracks > 0


def test_zero_field_config1():
    """Bz = 0: straight lines, a = 0 exactly (f04 = f24 = 0, q/pT never moves)."""
    import dataclasses
    b = generate_config(1)
    b0 = dataclasses.replace(b, geometry=dataclasses.replace(b.geometry, bz_kgauss=0.0))
    gpu = G.run_gpu(b0)
    ref = G.run_oracle(b0)
    G.compare(gpu, ref, b0.geometry.n_rows, rtol=RTOL)


def test_mirror_symmetries_on_the_gpu():
    """z -> -z (A side <-> C side) and y -> -y give the mirrored tracks, bit for bit, on the CUDA path itself."""
    import dataclasses
    b = generate_config(1)
    nr, ns = b.geometry.n_rows, b.geometry.n_sectors
    base = G.run_gpu(b, debug=False, debug_tracklets=False)

    def as_dict(g, remap=None, task_map=None):
        out = {}
        hb = g["track_hit_begin"].astype(np.int64)
        for t in range(g["n_tracks"]):
            h = g["hit_cluster"][hb[t]:hb[t] + int(g["track_nhits"][t])].astype(np.int64)
            if remap is not None:
                h = remap[h]
            task = int(g["track_task"][t])
            out[(task_map(task) if task_map else task, tuple(h.tolist()))] = t
        return out
    ref = as_dict(base)
    # z mirror: task s <-> s + 18 with identical (y, -z)
    counts = np.diff(b.row_offsets.astype(np.int64)).reshape(b.n_tasks, nr)
    src_task = (np.arange(b.n_tasks) + ns // 2) % ns
    offs = np.zeros(b.n_tasks * nr + 1, np.uint32)
    offs[1:] = np.cumsum(counts[src_task].ravel())
    idx = np.concatenate([np.arange(b.row_offsets[t * nr], b.row_offsets[(t + 1) * nr]) for t in src_task])
    mz = dataclasses.replace(b, y=b.y[idx], z=-b.z[idx], x=b.x[idx], row_offsets=offs)
    gz = G.run_gpu(mz, debug=False, debug_tracklets=False)
    dz = as_dict(gz, remap=idx, task_map=lambda t: (t + ns // 2) % ns)
    assert set(dz) == set(ref)
    sign_z = np.array([1, -1, 1, -1, 1], np.float32)
    for k, t in ref.items():
        assert np.array_equal(base["track_par"][:, t] * sign_z, gz["track_par"][:, dz[k]])
    # y mirror: sinphi and q/pT change sign
    gy = G.run_gpu(dataclasses.replace(b, y=-b.y), debug=False, debug_tracklets=False)
    dy = as_dict(gy)
    assert set(dy) == set(ref)
    sign_y = np.array([-1, 1, -1, 1, -1], np.float32)
    for k, t in ref.items():
        assert np.array_equal(base["track_par"][:, t] * sign_y, gy["track_par"][:, dy[k]])


def test_non_finite_clusters_do_not_hang_the_grid_build():
    """Outside the contract (R27: coordinates are finite) but it must come back: +-Inf and NaN clusters once made
    the coarsening loop of the grid build spin for ever.  They land in edge bins, pass no exact window test, and
    the rest of the event is tracked as the oracle tracks it."""
    b = generate_config(0)
    y, z = b.y.copy(), b.z.copy()
    rng = np.random.default_rng(3)
    noise = np.nonzero(b.truth_track < 0)[0]
    bad = rng.choice(noise, 12, replace=False)
    vals = [np.inf, -np.inf, np.nan]
    for k, i in enumerate(bad):
        if k % 2:
            y[i] = vals[k % 3]
        else:
            z[i] = vals[k % 3]
    import dataclasses
    bb = dataclasses.replace(b, y=y, z=z)
    gpu = G.run_gpu(bb)
    ref = G.run_oracle(bb)
    G.compare(gpu, ref, b.geometry.n_rows, rtol=RTOL)
    assert not (set(bad.tolist()) & set(gpu["hit_cluster"].tolist()))
    # a row made of NaN only
    geom = default_geometry(n_sectors=1, n_rows=12)
    pts = {(0, r): [(0.01 * float(geom.row_x[r]), 0.5 * float(geom.row_x[r]))] for r in range(12)}
    pts[(0, 5)] = [(float("nan"), float("nan"))] * 3
    gpu = G.run_gpu(batch_from_rows(geom, pts, n_tasks=1))
    assert gpu["status"] == 0


# ---- invariances on the GPU path ---------------------------------------------------------------
def test_batch_equals_single_events():
    """events on one GPU are independent - a batch of 3 gives the 3 single results."""
    evs = [generate_config(1), generate_config(1)]
    from tpc_workload.events import CONFIGS, generate_event
    evs[1] = generate_event(default_geometry(), CONFIGS[1]["spec"], 77, track_id_base=1_000_000)
    both = concat_batches(evs)
    gb = G.run_gpu(both, debug=False, debug_tracklets=False)
    base, tbase = 0, 0
    got = set()
    beg = gb["track_hit_begin"].astype(np.int64)
    for t in range(gb["n_tracks"]):
        got.add((int(gb["track_task"][t]), tuple(gb["hit_cluster"][beg[t]:beg[t] + int(gb["track_nhits"][t])].tolist())))
    want = set()
    for e in evs:
        g1 = G.run_gpu(e, debug=False, debug_tracklets=False)
        b1 = g1["track_hit_begin"].astype(np.int64)
        for t in range(g1["n_tracks"]):
            want.add((int(g1["track_task"][t]) + tbase,
                      tuple((g1["hit_cluster"][b1[t]:b1[t] + int(g1["track_nhits"][t])].astype(np.int64) + base).tolist())))
        base += e.n_clusters
        tbase += e.n_tasks
    assert got == want


def test_a_thousand_small_tasks_through_the_ordered_queue():
    """1000 single-sector events of 200 tracks in one call: more tracklets (about 170 k) than the device holds lanes,
    so the four a5 kernels draw them in diagonal order - here with few tracklets per task, i.e. a stagger of a tenth
    of a row per task and most tasks sharing the last offset, the opposite regime of config 3 (576 tasks of 2 200
    tracklets).  Every stage's debug output and every track must equal the oracle's; the queue order must not
    show in the result."""
    from tpc_workload.events import CONFIGS, generate_event
    geom = default_geometry(n_sectors=1)
    evs = [generate_event(geom, CONFIGS[0]["spec"], 5000 + i, track_id_base=i * 1_000_000) for i in range(1000)]
    b = concat_batches(evs)
    assert b.n_tasks == 1000
    gpu = G.run_gpu(b, debug=True, debug_tracklets=False)
    assert gpu["n_tracklets"] > 148 * 7 * 128, "the test is meant to exceed the lanes of every a5 kernel"
    ref = G.run_oracle(b, dump_tracklets=False)
    G.compare(gpu, ref, b.geometry.n_rows, rtol=RTOL, check_tracklets=False)


def test_result_independent_of_grid_bin_size():
    """SPEC 2: the grid is acceleration only."""
    b = generate_config(1)
    ref = G.run_oracle(b)
    for lo, hi in ((1.0, 5.0), (8.0, 50.0)):
        gpu = G.run_gpu(b, params_over=dict(grid_bin_min=lo, grid_bin_max=hi))
        G.compare(gpu, ref, b.geometry.n_rows, rtol=RTOL)


def test_run_to_run_determinism_including_track_order(cfg2):
    a = G.run_gpu(cfg2, debug=False, debug_tracklets=False)
    c = G.run_gpu(cfg2, debug=False, debug_tracklets=False)
    for k in ("track_task", "track_hit_begin", "track_nhits", "track_ndf", "track_x", "track_par", "track_cov",
              "track_chi2", "hit_cluster"):
        assert np.array_equal(a[k], c[k]), k


# ---- edge cases ---------------------------------------------------------------------------------
def test_empty_input_and_empty_tasks():
    geom = default_geometry(n_sectors=2)
    empty = batch_from_rows(geom, {}, n_tasks=2)
    gpu = G.run_gpu(empty)
    assert gpu["n_tracks"] == 0 and gpu["n_hits"] == 0 and gpu["status"] == 0 and gpu["n_tracklets"] == 0
    # config 0 event in task 2 of 4, the other tasks empty
    b0 = generate_config(0)
    g4 = default_geometry(n_sectors=1)
    nr = g4.n_rows
    offs = np.concatenate([np.zeros(2 * nr, np.uint32), b0.row_offsets, np.full(nr, b0.n_clusters, np.uint32)])
    import dataclasses
    b = dataclasses.replace(b0, n_tasks=4, row_offsets=offs)
    gpu = G.run_gpu(b)
    ref = G.run_oracle(b)
    G.compare(gpu, ref, nr, rtol=RTOL)
    assert set(gpu["track_task"].tolist()) == {2}


def test_hand_built_rows_ragged_and_ties():
    """Three straight tracks in a 12-row detector, one with duplicated clusters (equal chi2 ties broken
    by gid, SPEC 0), rows of 1..3 clusters."""
    geom = default_geometry(n_sectors=1, n_rows=12)
    pts = {}
    for r in range(12):
        x = float(geom.row_x[r])
        row = [(0.01 * x, 0.5 * x), (-0.02 * x, 0.2 * x)]
        if r % 2 == 0:
            row.append((0.01 * x, 0.5 * x))  # exact duplicate: tie
        if r >= 3:
            row.append((5.0 + 0.03 * x, 0.9 * x))
        pts[(0, r)] = row
    b = batch_from_rows(geom, pts, n_tasks=1)
    gpu = G.run_gpu(b)
    ref = G.run_oracle(b)
    G.compare(gpu, ref, 12, rtol=RTOL)
    assert ref.n_tracks >= 2


def test_rows_beyond_16_bit_indices():
    """Maximum sizes: three adjacent rows of 70 000 clusters each (row-local indices need more than 16 bits; bins
    hold ~17 clusters, so the candidate lists of the neighbour finder overflow and its serial search runs), next to
    ordinary rows with three straight tracks."""
    geom = default_geometry(n_sectors=1, n_rows=14)
    rng = np.random.default_rng(7)
    pts = {}
    for r in range(14):
        x = float(geom.row_x[r])
        row = [(0.01 * x, 0.5 * x), (-0.02 * x, 0.2 * x), (3.0 + 0.03 * x, 0.9 * x)]
        if 5 <= r <= 7:
            w = x * float(geom.tan_half_angle)
            yy = rng.uniform(-w, w, 70_000).astype(np.float32)
            zz = rng.uniform(0.0, 250.0, 70_000).astype(np.float32)
            row += list(zip(yy.tolist(), zz.tolist()))
        pts[(0, r)] = row
    b = batch_from_rows(geom, pts, n_tasks=1)
    assert int(np.diff(b.row_offsets.astype(np.int64)).max()) > 65535
    gpu = G.run_gpu(b, debug_tracklets=False)
    ref = G.run_oracle(b, dump_tracklets=False)
    G.compare(gpu, ref, 14, rtol=RTOL, check_tracklets=False)


def test_overflow_sets_status_and_never_writes_out_of_bounds():
    b = generate_config(0)
    ref = G.run_oracle(b)
    # tracklet capacity
    gpu = G.run_gpu(b, debug=False, debug_tracklets=False, max_tracklets=16)
    assert gpu["status"] & 1 and gpu["n_tracklets"] == 16
    # track capacity: totals are still reported, only the first slots are written
    gpu = G.run_gpu(b, debug=False, debug_tracklets=False, track_capacity=8)
    assert gpu["status"] & 2 and gpu["n_tracks"] == ref.n_tracks
    # hit capacity
    gpu = G.run_gpu(b, debug=False, debug_tracklets=False, hit_capacity=100)
    assert gpu["status"] & 4 and gpu["n_hits"] == len(ref.hit_cluster)


def test_host_buffer_entry_point_matches_device_entry_point():
    """tpc_track_batch_host (the e2e leg of bench.py) gives the same tracks as tpc_track_batch."""
    import torch
    from paper_1712_09434_b200 import Tracker
    b = generate_config(1)
    dev = torch.device("cuda:0")
    trk = Tracker(b.geometry, G.tracker_params_for(b))
    n = b.n_clusters
    y = torch.from_numpy(np.ascontiguousarray(b.y)).pin_memory()
    z = torch.from_numpy(np.ascontiguousarray(b.z)).pin_memory()
    ro = torch.from_numpy(b.row_offsets.astype(np.uint32).view(np.int32)).pin_memory()
    out = trk.alloc_outputs(n, dev, pinned_host=True)
    tcap, hcap = out.track_task.shape[0], out.hit_cluster.shape[0]
    ws = trk.alloc_workspace(trk.host_workspace_bytes(n, b.n_tasks, 0, tcap, hcap), dev)
    up, down = trk.track_batch_host(y, z, ro, b.n_tasks, out, ws)
    h = out.header.numpy()
    assert up == 8 * n + 4 * (b.n_tasks * b.geometry.n_rows + 1)
    assert down == 16 + 104 * int(h[0]) + 4 * int(h[1])  # 6 words + 5 par + 15 cov per track
    host = out.to_numpy()
    trk.close()
    ref = G.run_oracle(b, dump_tracklets=False)
    G.compare(host, ref, b.geometry.n_rows, rtol=RTOL, check_tracklets=False)


def test_host_entry_point_in_chunks_equals_one_call(cfg2):
    """A batch of more than 2^20 clusters goes through tpc_track_batch_host as three chunks of whole sector tasks on
    three streams (copies overlap kernels); the result must be the single call's, array for array."""
    import torch
    from paper_1712_09434_b200 import Tracker
    b = cfg2
    assert b.n_clusters > (1 << 20)
    dev = torch.device("cuda:0")
    ref = G.run_gpu(b, debug=False, debug_tracklets=False)
    trk = Tracker(b.geometry, G.tracker_params_for(b))
    n = b.n_clusters
    y = torch.from_numpy(np.ascontiguousarray(b.y)).pin_memory()
    z = torch.from_numpy(np.ascontiguousarray(b.z)).pin_memory()
    ro = torch.from_numpy(b.row_offsets.astype(np.uint32).view(np.int32)).pin_memory()
    out = trk.alloc_outputs(n, dev, pinned_host=True)
    tcap, hcap = out.track_task.shape[0], out.hit_cluster.shape[0]
    ws = trk.alloc_workspace(trk.host_workspace_bytes(n, b.n_tasks, 0, tcap, hcap), dev)
    for _ in range(2):  # twice: the streams and buffers of the chunks are reused
        up, down = trk.track_batch_host(y, z, ro, b.n_tasks, out, ws)
    host = out.to_numpy()
    trk.close()
    assert up == 8 * n + 4 * (b.n_tasks * b.geometry.n_rows + 3)  # y, z and the row offsets of three chunks (one end entry each)
    assert host["n_tracks"] == ref["n_tracks"] and host["n_hits"] == ref["n_hits"] and host["status"] == 0
    assert host["n_tracklets"] == ref["n_tracklets"]
    for k in ("track_task", "track_hit_begin", "track_nhits", "track_ndf", "track_x", "track_par", "track_cov",
              "track_chi2", "hit_cluster"):
        assert np.array_equal(host[k], ref[k]), k


def test_host_entry_point_in_chunks_overflow_is_reported(cfg2):
    """Capacities far too small, through the chunked host path: totals are still the true ones, status bits are
    set, only the first slots are written (and they are the single call's first tracks)."""
    import torch
    from paper_1712_09434_b200 import Tracker
    b = cfg2
    dev = torch.device("cuda:0")
    ref = G.run_gpu(b, debug=False, debug_tracklets=False)
    trk = Tracker(b.geometry, G.tracker_params_for(b))
    n = b.n_clusters
    y = torch.from_numpy(np.ascontiguousarray(b.y)).pin_memory()
    z = torch.from_numpy(np.ascontiguousarray(b.z)).pin_memory()
    ro = torch.from_numpy(b.row_offsets.astype(np.uint32).view(np.int32)).pin_memory()
    out = trk.alloc_outputs(n, dev, pinned_host=True, track_capacity=8, hit_capacity=100)
    ws = trk.alloc_workspace(trk.host_workspace_bytes(n, b.n_tasks, 0, 8, 100), dev)
    trk.track_batch_host(y, z, ro, b.n_tasks, out, ws)
    h = out.header.numpy()
    assert int(h[0]) == ref["n_tracks"] and int(h[1]) == ref["n_hits"] and int(h[3]) == ref["n_tracklets"]
    assert int(h[2]) & 2 and int(h[2]) & 4
    assert np.array_equal(out.track_task.numpy()[:8], ref["track_task"][:8])
    assert np.array_equal(out.track_nhits.numpy()[:8], ref["track_nhits"][:8])
    hb, nh = out.track_hit_begin.numpy()[:8].astype(np.int64), out.track_nhits.numpy()[:8].astype(np.int64)
    assert np.array_equal(hb, ref["track_hit_begin"][:8])
    for t in range(8):  # include/tpc_tracker.h: a track is valid iff its hits fit the hit capacity
        if hb[t] + nh[t] <= 100:
            assert np.array_equal(out.hit_cluster.numpy()[hb[t]:hb[t] + nh[t]], ref["hit_cluster"][hb[t]:hb[t] + nh[t]])
    trk.close()


def test_host_entry_point_chunks_with_one_heavy_task():
    """Chunk boundaries fall on whole tasks: a batch whose clusters sit almost all in one task leaves chunks empty.
    The chunked host path must still give the device path's result."""
    import torch
    from paper_1712_09434_b200 import Tracker
    geom = default_geometry(n_sectors=1, n_rows=20)
    rng = np.random.default_rng(11)
    pts = {}
    for r in range(20):
        x = float(geom.row_x[r])
        pts[(0, r)] = [(0.01 * x, 0.5 * x), (-0.02 * x, 0.2 * x)]
        pts[(3, r)] = [(0.02 * x, 0.3 * x)]
        w = x * float(geom.tan_half_angle)
        yy = rng.uniform(-w, w, 60_000).astype(np.float32)
        zz = rng.uniform(0.0, 250.0, 60_000).astype(np.float32)
        pts[(2, r)] = [(3.0 + 0.03 * x, 0.9 * x)] + list(zip(yy.tolist(), zz.tolist()))
    b = batch_from_rows(geom, pts, n_tasks=5)  # task 1 and 4 empty, task 2 holds 1.2 M clusters
    assert b.n_clusters > (1 << 20)
    dev = torch.device("cuda:0")
    ref = G.run_gpu(b, debug=False, debug_tracklets=False)
    trk = Tracker(b.geometry, G.tracker_params_for(b))
    n = b.n_clusters
    y = torch.from_numpy(np.ascontiguousarray(b.y)).pin_memory()
    z = torch.from_numpy(np.ascontiguousarray(b.z)).pin_memory()
    ro = torch.from_numpy(b.row_offsets.astype(np.uint32).view(np.int32)).pin_memory()
    out = trk.alloc_outputs(n, dev, pinned_host=True)
    ws = trk.alloc_workspace(trk.host_workspace_bytes(n, b.n_tasks, 0, out.track_task.shape[0], out.hit_cluster.shape[0]), dev)
    trk.track_batch_host(y, z, ro, b.n_tasks, out, ws)
    host = out.to_numpy()
    trk.close()
    assert host["n_tracks"] == ref["n_tracks"] and host["n_hits"] == ref["n_hits"] and host["status"] == ref["status"] == 0
    assert ref["n_tracks"] >= 4
    for k in ("track_task", "track_hit_begin", "track_nhits", "track_ndf", "track_x", "track_par", "track_cov",
              "track_chi2", "hit_cluster"):
        assert np.array_equal(host[k], ref[k]), k


def test_counters_match_the_oracle_counters():
    """The device counters feed the algorithmic-bytes formula of bench.py."""
    b = generate_config(1)
    gpu = G.run_gpu(b, counters=True)
    ref = G.run_oracle(b)
    c, o = gpu["counters"], ref.counters
    assert c["clusters"] == o["clusters"]
    assert c["start_hits"] == o["start_hits"]
    assert c["tracklets_built"] == o["tracklets_built"]
    assert c["tracklets_kept"] == o["tracklets_kept"]
    assert c["chain_hits"] == o["chain_hits"]
    assert c["searches"] == o["search_up"] + o["search_dn"]
    assert c["tracklet_hits"] == o["tracklet_hits"]
    assert c["row_steps"] == o["row_steps"]


def test_host_pipeline_two_batches_in_flight(cfg2):
    """tpc_host_submit / tpc_host_collect: two different batches in flight at once, several rounds; every collected
    result is the single device call's, array for array, and a slot cannot be reused before it is collected."""
    import torch
    from paper_1712_09434_b200 import Tracker, TpcError
    dev = torch.device("cuda:0")
    batches = [cfg2, generate_config(1)]
    refs = [G.run_gpu(b, debug=False, debug_tracklets=False) for b in batches]
    trk = Tracker(cfg2.geometry, G.tracker_params_for(cfg2))
    try:
        host, outs, wss = [], [], []
        for b in batches:
            n = b.n_clusters
            host.append((torch.from_numpy(np.ascontiguousarray(b.y)).pin_memory(),
                         torch.from_numpy(np.ascontiguousarray(b.z)).pin_memory(),
                         torch.from_numpy(b.row_offsets.astype(np.uint32).view(np.int32)).pin_memory()))
            out = trk.alloc_outputs(n, dev, pinned_host=True)
            outs.append(out)
            wss.append(trk.alloc_workspace(trk.host_workspace_bytes(n, b.n_tasks, 0, out.track_task.shape[0],
                                                                    out.hit_cluster.shape[0]), dev))

        def submit(k):
            y, z, ro = host[k]
            trk.host_submit(k, y, z, ro, batches[k].n_tasks, outs[k].track_task.shape[0], outs[k].hit_cluster.shape[0], wss[k])

        def check(k, up):
            b, ref, out = batches[k], refs[k], outs[k]
            assert up == 8 * b.n_clusters + 4 * (b.n_tasks * b.geometry.n_rows + 1)
            h = out.header.numpy()
            assert int(h[0]) == ref["n_tracks"] and int(h[1]) == ref["n_hits"] and int(h[2]) == 0
            nt, nh = ref["n_tracks"], ref["n_hits"]
            for f in ("track_task", "track_hit_begin", "track_nhits", "track_ndf", "track_x", "track_chi2"):
                assert np.array_equal(getattr(out, f).numpy()[:nt], ref[f]), f
            assert np.array_equal(out.track_par.numpy()[:, :nt], ref["track_par"])
            assert np.array_equal(out.track_cov.numpy()[:, :nt], ref["track_cov"])
            assert np.array_equal(out.hit_cluster.numpy()[:nh], ref["hit_cluster"])

        submit(0)
        with pytest.raises(TpcError):
            submit(0)                       # not collected yet
        for _ in range(3):
            submit(1)
            up, down = trk.host_collect(0, outs[0]); check(0, up)
            submit(0)
            up, down = trk.host_collect(1, outs[1]); check(1, up)
        up, down = trk.host_collect(0, outs[0]); check(0, up)
        assert down > 4 * refs[0]["n_hits"]
        with pytest.raises(TpcError):
            trk.host_collect(0, outs[0])    # nothing in flight
    finally:
        trk.close()
