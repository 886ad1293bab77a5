"""Pins of the whole oracle path (docs/ARITH_SPEC.md sections 2-7) - CPU only.

Nothing here re-types the oracle's sequence.  The neighbour finder is pinned by
the exhaustive search and by hand-computed chi2 values; cleaner / start hits by
their post-conditions; the Kalman fit by noiseless-helix recovery (fp64, 1e-5),
a weighted linear regression (Bz = 0) and unit pulls; selector and output by
uniqueness invariants and a hand-built overlap; the system by batch, grid-size
and mirror invariances (PAPER.md L138 sectors independent, L127 events
independent, L182 <= 159 clusters per track, L121 seeds of 5-10 hits).
"""
import dataclasses
import json
import os

import numpy as np
import pytest

import oracle
from oracle import OracleParams
from helpers import batch_from_rows, single_track_events, tracks_as_dict
from tpc_workload import (default_geometry, generate_config, generate_tracks_event, concat_batches, take_tasks)

GOLDEN = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_facts.json")))


def run(b, **kw):
    return oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, **kw)


@pytest.fixture(scope="module")
def cfg0():
    b = generate_config(0)
    return b, run(b)


@pytest.fixture(scope="module")
def cfg1():
    b = generate_config(1)
    return b, run(b)


# ---------------------------------------------------------------- neighbour finder
def test_links_equal_exhaustive_search(cfg0, cfg1):
    """SPEC 3 is defined as a search over ALL (u,d) pairs; the grid must not change it."""
    for b, res in (cfg0, cfg1):
        brute = run(b, brute_force_neighbours=True)
        np.testing.assert_array_equal(res.link_up, brute.link_up)
        np.testing.assert_array_equal(res.link_dn, brute.link_dn)
        assert (res.link_up >= 0).sum() > 0.8 * b.n_clusters


def test_links_hand_built_three_rows():
    """Row spacing is uniform, so chi2 = (dx*(yu+yd-2y))^2*wy + (dx*(zu+zd-2z))^2*wz (R3)."""
    g = default_geometry(n_sectors=1)
    dx = float(g.row_x[11] - g.row_x[10])
    assert float(g.row_x[10] - g.row_x[9]) == dx  # holds for these rows in fp32
    # centre (0, 100) in row 10; ups in row 11, downs in row 9.
    pts = {
        (0, 10): [(0.0, 100.0)],
        (0, 11): [(0.30, 101.0), (0.10, 101.1), (1.9, 101.0), (2.1, 101.0)],
        (0, 9): [(-0.12, 99.0), (-0.30, 98.9), (0.0, 97.0)],
    }
    b = batch_from_rows(g, pts)
    res = run(b)
    # gids: row 9 -> 0,1,2 ; row 10 -> 3 ; row 11 -> 4,5,6,7
    wy, wz = 1 / 0.1 ** 2, 1 / 0.15 ** 2
    best = None
    for u, (yu, zu) in zip((4, 5, 6, 7), pts[(0, 11)]):
        if abs(yu - 0.0) > 2.0 or abs(zu - 100.0 * g.row_x[11] / g.row_x[10]) > 1.5:
            continue
        for d, (yd, zd) in zip((0, 1, 2), pts[(0, 9)]):
            if abs(yd) > 2.0 or abs(zd - 100.0 * g.row_x[9] / g.row_x[10]) > 1.5:
                continue
            chi = (dx * (yu + yd)) ** 2 * wy + (dx * (zu + zd - 200.0)) ** 2 * wz
            if chi < 75 and (best is None or chi < best[0]):
                best = (chi, u, d)
    # by hand: (4,1) has second differences (0.30-0.30, 101.0+98.9-200) = (0, -0.1) -> chi2 = (dx*0.1)^2*wz = 0.467;
    # (5,0) has (-0.02, 0.1) -> 0.042 + 0.467: slightly worse
    assert best[1:] == (4, 1)
    assert res.link_up[3] == 4 and res.link_dn[3] == 1
    # rows without both neighbours: no links (R5, pair or nothing)
    assert (res.link_up[[0, 1, 2, 4, 5, 6, 7]] == -1).all() and (res.link_dn[[0, 1, 2, 4, 5, 6, 7]] == -1).all()


def test_links_window_chi2_cut_and_ties():
    g = default_geometry(n_sectors=1)
    r = 50
    zr_u, zr_d = g.row_x[r + 1] / g.row_x[r], g.row_x[r - 1] / g.row_x[r]
    z = 80.0
    # straight line through the origin in z, exact duplicates in the up row -> tie broken by smaller gid
    pts = {(0, r - 1): [(0.0, z * zr_d)], (0, r): [(0.0, z)], (0, r + 1): [(0.0, z * zr_u), (0.0, z * zr_u)]}
    res = run(batch_from_rows(g, pts))
    assert res.link_up[1] == 2 and res.link_dn[1] == 0
    # chi2 cut: kink of 1.0 cm in y over 1.025 cm rows -> chi2 = (dx*1.0)^2/0.01 = 105 > 75
    pts = {(0, r - 1): [(0.0, z * zr_d)], (0, r): [(0.0, z)], (0, r + 1): [(1.0, z * zr_u)]}
    res = run(batch_from_rows(g, pts))
    assert res.link_up[1] == -1 and res.link_dn[1] == -1
    # 0.8 cm kink -> chi2 = 67 < 75: linked
    pts[(0, r + 1)] = [(0.8, z * zr_u)]
    res = run(batch_from_rows(g, pts))
    assert res.link_up[1] == 2 and res.link_dn[1] == 0
    # window: z of the up hit 1.6 cm off the projected z -> not a candidate even though chi2 would pass loosely
    pts[(0, r + 1)] = [(0.0, z * zr_u + 1.6)]
    prm = OracleParams(nf_chi2_max=1e9)
    res = oracle.track(g, *(lambda b: (b.y, b.z, b.row_offsets, b.n_tasks))(batch_from_rows(g, pts)), params=prm)
    assert res.link_up[1] == -1
    pts[(0, r + 1)] = [(0.0, z * zr_u + 1.4)]
    res = oracle.track(g, *(lambda b: (b.y, b.z, b.row_offsets, b.n_tasks))(batch_from_rows(g, pts)), params=prm)
    assert res.link_up[1] == 2


# ---------------------------------------------------------------- cleaner, start hits, chains
def test_cleaner_postconditions(cfg0, cfg1):
    for b, res in (cfg0, cfg1):
        cu, cd = res.clean_up, res.clean_dn
        h = np.nonzero(cu >= 0)[0]
        np.testing.assert_array_equal(cd[cu[h]], h)          # cu[h]=u  =>  cd[u]=h
        h = np.nonzero(cd >= 0)[0]
        np.testing.assert_array_equal(cu[cd[h]], h)
        # cleaned links are a subset of raw links
        assert ((cu == res.link_up) | (cu == -1)).all() and ((cd == res.link_dn) | (cd == -1)).all()
        # a mutual raw link survives
        h = np.nonzero(res.link_up >= 0)[0]
        mutual = res.link_dn[res.link_up[h]] == h
        np.testing.assert_array_equal(cu[h] >= 0, mutual)
        # links go to the adjacent row of the same task
        tr = np.repeat(np.arange(len(b.row_offsets) - 1), np.diff(b.row_offsets.astype(np.int64)))
        h = np.nonzero(cu >= 0)[0]
        np.testing.assert_array_equal(tr[cu[h]], tr[h] + 1)


def test_start_hits_one_per_chain(cfg0, cfg1):
    for b, res in (cfg0, cfg1):
        cu, cd = res.clean_up, res.clean_dn
        expect = np.nonzero((cu >= 0) & (cd < 0))[0]
        np.testing.assert_array_equal(res.start_hits, expect.astype(np.uint32))
        # chains are vertex-disjoint paths: walking up from every start hit visits each linked cluster once
        seen = np.zeros(b.n_clusters, np.int32)
        lens = []
        for h0 in res.start_hits:
            n, h = 0, int(h0)
            while h >= 0:
                seen[h] += 1
                n += 1
                h = int(cu[h])
            lens.append(n)
        assert seen.max() == 1
        assert (seen[(cu >= 0) | (cd >= 0)] == 1).all()
        lens = np.array(lens)
        assert res.counters["tracklets_built"] == int((lens >= 5).sum())  # S3, lower end of L121's 5-10 hits
        assert res.counters["tracklets_built"] == res.n_tracklets


# ---------------------------------------------------------------- Kalman fit / following
def test_noiseless_helices_recovered_fp64():
    """north_star: every cluster collected, fitted parameters = truth to 1e-5 (fp64 instantiation)."""
    rng = np.random.default_rng(11)
    b = single_track_events(80, rng, pt_range=(0.3, 5.0), sigma_y=0.0, sigma_z=0.0)
    # the generator's exact fp64 crossings (truth_state) are the input: no fp32 rounding of y, z
    res = oracle.track(b.geometry, b.truth_state[:, 0].copy(), b.truth_state[:, 1].copy(), b.row_offsets, b.n_tasks,
                       precision="f64")
    _check_recovery(b, res, rtol=1e-5, short_sigma_frac=2e-3)


def test_noiseless_helices_recovered_fp32():
    """the fp32 instantiation reaches ~2e-5 on long legs; held to 1e-4."""
    rng = np.random.default_rng(11)
    b = single_track_events(80, rng, pt_range=(0.3, 5.0), sigma_y=0.0, sigma_z=0.0)
    res = run(b)
    _check_recovery(b, res, rtol=1e-4, short_sigma_frac=2e-2)


def _check_recovery(b, res, rtol, short_sigma_frac):
    """SURVEY 8(c) 'Whole O5': EVERY leg with >= MIN_HITS (10) rows and |sin phi| < 0.95 is collected with every
    cluster, exactly once.  Parameters: legs of >= 40 rows equal the truth to rtol; shorter fragments (10..39 rows:
    sector-crossing stubs, sigma(q/pT) > 1 c/GeV) are held to short_sigma_frac of their OWN fitted error instead -
    the turn-around keeps 1/turn_cov_scale = 1 % of the up pass's estimate (K4, reading R15: scale, do not
    re-initialise), and on a 10-row lever arm that estimate still carries the q = 0 linearisation of the seed:
    measured fp64 2.7e-3 relative = 1e-3 sigma on 10..19 rows, 7e-5 on 20..39, 2.8e-6 on 40..79, 8e-7 beyond
    (D10)."""
    nr = b.geometry.n_rows
    tr = np.repeat(np.arange(len(b.row_offsets) - 1), np.diff(b.row_offsets.astype(np.int64)))
    task_of, row_of = tr // nr, tr % nr
    n_long, n_short = 0, 0
    tracks_by_task = {}
    for t in range(res.n_tracks):
        tracks_by_task.setdefault(int(res.track_task[t]), []).append(t)
    for task in np.unique(task_of):
        for leg in (0, 1):
            sel = np.nonzero((task_of == task) & (b.truth_leg == leg))[0]
            if len(sel) < 10 or np.abs(b.truth_state[sel, 2]).max() >= 0.95:
                continue
            cand = [t for t in tracks_by_task.get(int(task), []) if set(res.track_hits(t)) == set(sel)]
            assert len(cand) == 1, f"task {task} leg {leg} ({len(sel)} rows): clusters not collected exactly once"
            t = cand[0]
            first = sel[np.argmin(row_of[sel])]
            truth = b.truth_state[first].copy()
            got = res.track_par[:, t].astype(np.float64)
            assert float(res.track_x[t]) == float(b.geometry.row_x[row_of[first]])
            if len(sel) >= 40:
                scale = np.array([max(abs(truth[0]), 1.0), max(abs(truth[1]), 1.0), 1.0, 1.0, max(abs(truth[4]), 1.0)])
                np.testing.assert_array_less(np.abs(got - truth) / scale, rtol)
                n_long += 1
            else:
                sig = np.sqrt(res.track_cov[[0, 2, 5, 9, 14], t].astype(np.float64))
                np.testing.assert_array_less(np.abs(got - truth), short_sigma_frac * sig)
                n_short += 1
    assert n_long >= 80 and n_short >= 8


def test_fit_equals_weighted_linear_regression_when_bz_zero():
    """Bz = 0: transport is a straight line, so y(x) and z(l) fits are weighted regressions (fp64)."""
    g = dataclasses.replace(default_geometry(), bz_kgauss=0.0)
    rng = np.random.default_rng(5)
    evs = []
    for e in range(12):
        evs.append(generate_tracks_event(g, [1.0], [1.0], rng.uniform(0, 2 * np.pi, 1), rng.uniform(-0.8, 0.8, 1),
                                         [0.0], 0.1, 0.15, 0.0, rng))
    b = concat_batches(evs)
    res = oracle.track(g, b.y.astype(np.float64), b.z.astype(np.float64), b.row_offsets, b.n_tasks, precision="f64")
    nr = g.n_rows
    tr = np.repeat(np.arange(len(b.row_offsets) - 1), np.diff(b.row_offsets.astype(np.int64)))
    assert res.n_tracks >= 10
    for t in range(res.n_tracks):
        hits = res.track_hits(t).astype(np.int64)
        if len(hits) < 60:
            continue
        X = g.row_x[tr[hits] % nr].astype(np.float64)
        Y, Z = b.y[hits].astype(np.float64), b.z[hits].astype(np.float64)
        x0 = float(res.track_x[t])
        assert x0 == X.min()
        A = np.stack([np.ones_like(X), X - x0], 1)
        (y0, slope), *_ = np.linalg.lstsq(A, Y, rcond=None)
        s = slope / np.sqrt(1 + slope * slope)
        par = res.track_par[:, t]
        sig = np.sqrt(res.track_cov[[0, 2, 5, 9], t])
        # The prior is diffuse (C0, then x100 at the turn-around, SPEC K4) and the down pass re-fits every hit, so
        # the estimate is the regression's up to ~1 % of the linearisation error: within 0.01 sigma of each parameter.
        assert abs(par[0] - y0) < 0.01 * sig[0] and abs(par[2] - s) < 0.01 * sig[2]
        ell = (X - x0) * np.sqrt(1 + slope * slope)
        (z0, tz), *_ = np.linalg.lstsq(np.stack([np.ones_like(ell), ell], 1), Z, rcond=None)
        assert abs(par[1] - z0) < 0.01 * sig[1] and abs(par[3] - tz) < 0.01 * sig[3]
        # ... and its covariance is the regression's (normal equations), within the 1 % prior weight
        cov_y = 0.1 ** 2 * np.linalg.inv(A.T @ A)
        Az = np.stack([np.ones_like(ell), ell], 1)
        cov_z = 0.15 ** 2 * np.linalg.inv(Az.T @ Az)
        assert abs(sig[0] ** 2 / cov_y[0, 0] - 1) < 0.02 and abs(sig[1] ** 2 / cov_z[0, 0] - 1) < 0.02
        assert abs(sig[3] ** 2 / cov_z[1, 1] - 1) < 0.02
        ds_dslope = (1 + slope * slope) ** -1.5
        assert abs(sig[2] ** 2 / (cov_y[1, 1] * ds_dslope ** 2) - 1) < 0.02
        # q/pT is unconstrained without a field: stays at its seed value 0 with the (scaled) prior variance
        assert par[4] == 0.0
        assert res.track_ndf[t] == 2 * len(hits) - 5


@pytest.mark.parametrize("bz,prec,n_ev", [(5.0, "f32", 4000), (5.0, "f64", 2000), (0.0, "f32", 2000)])
def test_unit_pulls(bz, prec, n_ev):
    """north_star / SURVEY 8(c): the Kalman fit of straight lines and helices has unbiased, unit-width pulls:
    |mean| < 0.05, width 1 +- 0.1, on thousands of tracks (statistical error of a mean over 2000: 0.022)."""
    g = dataclasses.replace(default_geometry(), bz_kgauss=bz)
    rng = np.random.default_rng(21)
    b = single_track_events(n_ev, rng, pt_range=(0.4, 5.0), geom=g)
    dt = np.float32 if prec == "f32" else np.float64
    res = oracle.track(g, b.y.astype(dt), b.z.astype(dt), b.row_offsets, b.n_tasks, precision=prec)
    nr = g.n_rows
    tr = np.repeat(np.arange(len(b.row_offsets) - 1), np.diff(b.row_offsets.astype(np.int64)))
    pulls, chi = [], []
    diag = [0, 2, 5, 9, 14]
    for t in range(res.n_tracks):
        hits = res.track_hits(t).astype(np.int64)
        if len(hits) < 40 or len(set(b.truth_track[hits])) != 1:
            continue
        first = hits[0]
        assert (np.diff(tr[hits]) > 0).all()  # ascending rows (L3)
        truth = b.truth_state[first]
        par = res.track_par[:, t].astype(np.float64)
        var = res.track_cov[diag, t].astype(np.float64)
        assert (var > 0).all()
        pulls.append((par - truth) / np.sqrt(var))
        chi.append(float(res.track_chi2[t]) / int(res.track_ndf[t]))
    pulls = np.array(pulls)
    assert len(pulls) > 0.9 * n_ev
    n_par = 5 if bz != 0.0 else 4  # q/pT has no information at Bz = 0
    for j in range(n_par):
        assert abs(pulls[:, j].mean()) < 0.05, (j, pulls[:, j].mean())
        assert abs(pulls[:, j].std() - 1.0) < 0.1, (j, pulls[:, j].std())
    assert abs(np.mean(chi) - 1.0) < 0.02


# ---------------------------------------------------------------- selector / output
def test_output_invariants(cfg0, cfg1):
    for b, res in (cfg0, cfg1):
        nr = b.geometry.n_rows
        tr = np.repeat(np.arange(len(b.row_offsets) - 1), np.diff(b.row_offsets.astype(np.int64)))
        assert len(np.unique(res.hit_cluster)) == len(res.hit_cluster)          # a cluster is in <= 1 track
        assert res.track_nhits.min() >= 10 and res.track_nhits.max() <= GOLDEN["max_clusters_per_track"]["value"]
        np.testing.assert_array_equal(res.track_hit_begin, np.cumsum(res.track_nhits) - res.track_nhits)
        for t in range(res.n_tracks):
            h = res.track_hits(t).astype(np.int64)
            assert (tr[h] // nr == res.track_task[t]).all()
            assert (np.diff(tr[h] % nr) > 0).all()                                # <= 1 hit per row, ascending
            assert res.track_x[t] <= b.geometry.row_x[tr[h[0]] % nr]
        # efficiency sanity (parity unpinned): most long true legs are found
        eff_hits = len(res.hit_cluster) / (b.truth_track >= 0).sum()
        assert eff_hits > 0.9


def test_selector_resolves_shared_clusters_hand_built():
    """Two straight tracks crossing in y: longer tracklet owns the shared clusters (R16)."""
    g = dataclasses.replace(default_geometry(n_sectors=1), bz_kgauss=0.0)
    rng = np.random.default_rng(3)
    # track A: rows 0..158, track B: crosses A around row 80 in y at the same z slope
    pts = {}
    for r in range(159):
        x = float(g.row_x[r])
        pts[(0, r)] = [(0.02 * (x - 166.0), 0.5 * x)]
        if 40 <= r <= 120:
            pts[(0, r)].append((-0.02 * (x - 166.0), 0.5 * x))
    b = batch_from_rows(g, pts)
    res = run(b, dump_tracklets=True)
    assert len(np.unique(res.hit_cluster)) == len(res.hit_cluster)
    # key = (nHits << 32) | (~h0): recompute owners from the tracklet dump and compare with the output
    owner = {}
    for i in range(res.n_tracklets):
        n = int(res.tracklet_nhits[i])
        if n < 10:
            continue
        key = (n << 32) | (0xFFFFFFFF - int(res.tracklet_start[i]))
        for h in res.tracklet_map[i]:
            if h >= 0:
                owner[int(h)] = max(owner.get(int(h), 0), key)
    expect = set()
    for i in range(res.n_tracklets):
        n = int(res.tracklet_nhits[i])
        key = (n << 32) | (0xFFFFFFFF - int(res.tracklet_start[i]))
        kept = tuple(int(h) for h in res.tracklet_map[i] if h >= 0 and owner.get(int(h)) == key)
        if n >= 10 and len(kept) >= 10:
            expect.add(kept)
    got = {tuple(int(h) for h in res.track_hits(t)) for t in range(res.n_tracks)}
    assert got == expect and len(got) >= 2
    assert res.track_nhits.max() >= 150  # the long track is complete


# ---------------------------------------------------------------- system invariances
def _compare_results(a, b_, map_b_to_a=None, par_rtol=0.0):
    da, db = tracks_as_dict(a), tracks_as_dict(b_)
    if map_b_to_a is not None:
        db = {(k[0], tuple(int(map_b_to_a[h]) for h in k[1])): v for k, v in db.items()}
    assert set(da) == set(db)
    for k, ta in da.items():
        tb = db[k]
        if par_rtol == 0.0:
            np.testing.assert_array_equal(a.track_par[:, ta], b_.track_par[:, tb])
            np.testing.assert_array_equal(a.track_cov[:, ta], b_.track_cov[:, tb])


def test_grid_size_independence(cfg0):
    b, res = cfg0
    for lo, hi in ((1.0, 5.0), (8.0, 50.0)):
        r2 = run(b, params=OracleParams(grid_bin_min=lo, grid_bin_max=hi))
        np.testing.assert_array_equal(res.link_up, r2.link_up)
        np.testing.assert_array_equal(res.link_dn, r2.link_dn)
        _compare_results(res, r2)


def test_tasks_are_independent(cfg1):
    """PAPER.md L138 / L127: a sector task tracked alone gives what it gives inside the batch."""
    b, res = cfg1
    full = tracks_as_dict(res)
    for tasks in ([3], [20, 21], list(range(0, 36, 5))):
        sub, sel = take_tasks(b, tasks)
        rs = run(sub)
        got = {(k[0], tuple(int(sel[h]) for h in k[1])) for k in tracks_as_dict(rs)}
        want = {k for k in full if k[0] in tasks}
        assert got == want and len(want) > 0


def test_batch_of_events_equals_single_events():
    evs = [generate_config(1) for _ in range(1)]
    rng = np.random.default_rng(9)
    g = default_geometry()
    evs = [generate_tracks_event(g, np.exp(rng.uniform(np.log(0.2), np.log(5), 150)),
                                 np.where(rng.random(150) < 0.5, -1.0, 1.0), rng.uniform(0, 2 * np.pi, 150),
                                 rng.uniform(-0.9, 0.9, 150), np.zeros(150), 0.1, 0.15, 0.02, rng,
                                 track_id_base=1000 * e) for e in range(3)]
    batch = concat_batches(evs)
    rb = run(batch)
    got = set(tracks_as_dict(rb))
    want, base = set(), 0
    for e, ev in enumerate(evs):
        r1 = run(ev)
        want |= {(k[0] + 36 * e, tuple(h + base for h in k[1])) for k in tracks_as_dict(r1)}
        base += ev.n_clusters
    assert got == want and len(want) > 200


def _mirror_z(b):
    """z -> -z swaps the A and C side: task s <-> s+18 with identical (y, -z)."""
    nr, ns = b.geometry.n_rows, b.geometry.n_sectors
    counts = np.diff(b.row_offsets.astype(np.int64)).reshape(b.n_tasks, nr)
    src_task = (np.arange(b.n_tasks) + ns // 2) % ns
    new_counts = counts[src_task]
    offs = np.zeros(b.n_tasks * nr + 1, np.uint32)
    offs[1:] = np.cumsum(new_counts.ravel())
    idx = np.concatenate([np.arange(b.row_offsets[t * nr], b.row_offsets[(t + 1) * nr]) for t in src_task])
    return dataclasses.replace(b, y=b.y[idx], z=-b.z[idx], x=b.x[idx], row_offsets=offs), idx


def test_mirror_symmetries(cfg1):
    b, res = cfg1
    ns = b.geometry.n_sectors
    # z mirror
    m, idx = _mirror_z(b)
    rm = run(m)
    got = {((k[0] + ns // 2) % ns, tuple(int(idx[h]) for h in k[1])): v for k, v in tracks_as_dict(rm).items()}
    ref = tracks_as_dict(res)
    assert set(got) == set(ref)
    sign_z = np.array([1, -1, 1, -1, 1], np.float32)
    for k, t in ref.items():
        np.testing.assert_array_equal(res.track_par[:, t] * sign_z, rm.track_par[:, got[k]])
    # y mirror (y -> -y, curvature flips): same tracks with sinphi, q/pT negated
    my = dataclasses.replace(b, y=-b.y)
    ry = run(my)
    goty = tracks_as_dict(ry)
    assert set(goty) == set(ref)
    sign_y = np.array([-1, 1, -1, 1, -1], np.float32)
    for k, t in ref.items():
        np.testing.assert_array_equal(res.track_par[:, t] * sign_y, ry.track_par[:, goty[k]])


def test_empty_and_degenerate_inputs():
    g = default_geometry()
    e = np.zeros(0, np.float32)
    res = oracle.track(g, e, e, np.zeros(36 * 159 + 1, np.uint32), 36)
    assert res.n_tracks == 0 and len(res.start_hits) == 0
    # clusters only in rows 0 and 158: no links at all (R21)
    pts = {(0, 0): [(0.0, 10.0)] * 3, (0, 158): [(0.0, 10.0)] * 3}
    res = run(batch_from_rows(default_geometry(n_sectors=1), pts))
    assert (res.link_up == -1).all() and res.n_tracks == 0
