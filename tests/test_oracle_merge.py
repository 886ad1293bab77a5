"""Pins of SPEC 9 (sector-segment merger + final refit, PAPER.md L138 / L140) on the CPU oracle.

Nothing here re-types the oracle's formulas: the rotation is checked against plain trigonometry in GLOBAL
coordinates and against finite differences of the closed-form helix, the merger against generator truth
(noiseless tracks that cross one and two sector boundaries), the refit against truth and by its pulls.
"""
from __future__ import annotations

import types

import numpy as np
import pytest

import oracle
from tpc_workload import default_geometry, generate_tracks_event, concat_batches
from helpers import A_PER_KG, helix_closed_form, unpack_cov, pack_cov

GEOM = default_geometry()
A = A_PER_KG * GEOM.bz_kgauss
ALPHA = 2.0 * np.pi / 18.0
X = GEOM.row_x.astype(np.float64)


def sector_angle(k):
    return (k % 18 + 0.5) * ALPHA


def to_global(k, x, p):
    """Point and direction angle of a local state of sector k, in global coordinates."""
    al = sector_angle(k)
    gx = x * np.cos(al) - p[0] * np.sin(al)
    gy = x * np.sin(al) + p[0] * np.cos(al)
    return gx, gy, al + np.arcsin(p[2])


def from_global(k, gx, gy, psi, z, t, q):
    al = sector_angle(k)
    return gx * np.cos(al) + gy * np.sin(al), np.array([-gx * np.sin(al) + gy * np.cos(al), z, np.sin(psi - al), t, q])


def rand_state(rng):
    x = rng.uniform(85, 247)
    p = np.array([rng.uniform(-0.17, 0.17) * x, rng.uniform(-240, 240), rng.uniform(-0.6, 0.6), rng.uniform(-1, 1),
                  rng.uniform(-3, 3)])
    return x, p


def rand_cov(rng):
    m = rng.normal(size=(5, 5)) * np.array([0.1, 0.15, 0.01, 0.01, 0.05])[:, None]
    return m @ m.T + np.diag([1e-4, 1e-4, 1e-6, 1e-6, 1e-5])


@pytest.mark.parametrize("d", [+1, -1])
def test_rotate_is_the_same_track_in_the_neighbours_frame(d):
    """R2, R4: point and direction through global coordinates (plain trigonometry), all 18 sectors incl. the wrap."""
    rng = np.random.default_rng(5)
    for k in range(18):
        for _ in range(20):
            x, p = rand_state(rng)
            ok, x1, p1, _ = oracle.rotate(x, p, pack_cov(np.eye(5)), d, 36, A)
            assert ok
            gx, gy, psi = to_global(k, x, p)
            x_ref, p_ref = from_global(k + d, gx, gy, psi, p[1], p[3], p[4])
            assert abs(x1 - x_ref) < 1e-10 and np.allclose(p1, p_ref, atol=1e-10, rtol=0)


def test_rotate_there_and_back_is_the_identity():
    rng = np.random.default_rng(6)
    for _ in range(100):
        x, p = rand_state(rng)
        c = pack_cov(rand_cov(rng))
        ok1, x1, p1, c1 = oracle.rotate(x, p, c, +1, 36, A)
        ok2, x2, p2, c2 = oracle.rotate(x1, p1, c1, -1, 36, A)
        assert ok1 and ok2
        assert abs(x2 - x) < 1e-10 and np.allclose(p2, p, atol=1e-10, rtol=0)
        assert np.allclose(c2, c, rtol=1e-8, atol=1e-14)


def test_rotate_fails_beyond_the_angle_limit_and_leaves_the_state():
    c = pack_cov(np.eye(5))
    p = np.array([3.0, 10.0, 0.80, 0.2, 0.5])        # sin(phi - 20 deg) fine, sin(phi + 20 deg) = 0.957 > 0.95
    ok, x1, p1, c1 = oracle.rotate(120.0, p, c, -1, 36, A)  # d = -1 turns the frame by -alpha: phi' = phi + alpha
    assert not ok and x1 == 120.0 and np.array_equal(p1, p) and np.array_equal(c1, c)
    ok, _, p2, _ = oracle.rotate(120.0, p, c, +1, 36, A)
    assert ok and abs(p2[2] - np.sin(np.arcsin(0.80) - ALPHA)) < 1e-12


@pytest.mark.parametrize("d", [+1, -1])
def test_rotate_covariance_is_J_C_Jt_with_the_finite_difference_jacobian(d):
    """R5..R7.  J is taken numerically: perturb the state at the old x, express every perturbed track at the
    NOMINAL new x (rotate through global coordinates, then the closed-form helix back to that x)."""
    rng = np.random.default_rng(7)
    for _ in range(20):
        x, p = rand_state(rng)
        k = int(rng.integers(0, 18))

        def image(pp, x_nom=None):
            gx, gy, psi = to_global(k, x, pp)
            xr, pr = from_global(k + d, gx, gy, psi, pp[1], pp[3], pp[4])
            return xr, pr if x_nom is None else helix_closed_form(xr, pr, x_nom, A)
        x_nom, p_nom = image(p)
        J = np.zeros((5, 5))
        for j in range(5):
            h = 1e-6 * max(1.0, abs(p[j]))
            pp, pm = p.copy(), p.copy()
            pp[j] += h; pm[j] -= h
            J[:, j] = (image(pp, x_nom)[1] - image(pm, x_nom)[1]) / (2 * h)
        C = rand_cov(rng)
        ok, x1, p1, c1 = oracle.rotate(x, p, pack_cov(C), d, 36, A)
        assert ok and abs(x1 - x_nom) < 1e-10
        ref = J @ C @ J.T
        scale = np.sqrt(np.outer(np.diag(ref), np.diag(ref)))
        assert np.max(np.abs(unpack_cov(c1) - ref) / scale) < 2e-6


# ---- merger + refit against generator truth -------------------------------------------------------
def crossing_events(n, rng, sigma_y, sigma_z, pt_range=(0.25, 1.5)):
    evs = []
    for e in range(n):
        pt = np.exp(rng.uniform(np.log(pt_range[0]), np.log(pt_range[1]), 1))
        ch = np.where(rng.random(1) < 0.5, -1.0, 1.0)
        ph = rng.uniform(0, 2 * np.pi, 1)
        et = rng.uniform(-0.9, 0.9, 1)
        evs.append(generate_tracks_event(GEOM, pt, ch, ph, et, np.zeros(1), sigma_y, sigma_z, 0.0, rng,
                                         track_id_base=e * 10))
    return concat_batches(evs)


def leg0_segments(b, ev):
    """[(sector, gids sorted by row)] of the outgoing leg of the one track of event ev, innermost sector first."""
    nr, ns = b.geometry.n_rows, b.geometry.n_sectors
    lo, hi = int(b.row_offsets[ev * ns * nr]), int(b.row_offsets[(ev + 1) * ns * nr])
    g = np.arange(lo, hi)
    g = g[b.truth_leg[lo:hi] == 0]
    tr = np.searchsorted(b.row_offsets, g, side="right") - 1
    sec, row = (tr // nr) % ns, tr % nr
    segs = []
    for s in np.unique(sec):
        m = sec == s
        segs.append((int(s), g[m][np.argsort(row[m])], np.sort(row[m])))
    segs.sort(key=lambda t: t[2][0])
    return segs


def test_noiseless_crossing_tracks_are_merged_with_every_cluster_and_refitted_to_truth():
    """north_star-style pin for SPEC 9: tracks that cross one and two sector boundaries come out as ONE merged
    track holding every cluster, and the refit equals truth to 1e-5 (fp64 instantiation)."""
    rng = np.random.default_rng(11)
    b = crossing_events(260, rng, 0.0, 0.0)
    prm = oracle.OracleParams()
    # the generator's exact fp64 crossings (truth_state) are the input: no fp32 rounding of y, z
    y64, z64 = b.truth_state[:, 0].copy(), b.truth_state[:, 1].copy()
    res = oracle.track(b.geometry, y64, z64, b.row_offsets, b.n_tasks, params=prm, precision="f64")
    m = oracle.merge_refit(b.geometry, y64, z64, b.row_offsets, b.n_tasks, res, params=prm, precision="f64")
    ns = b.geometry.n_sectors
    first_gid = res.hit_cluster[res.track_hit_begin.astype(np.int64)]
    n_by_seg = {2: 0, 3: 0}
    for ev in range(b.n_events):
        segs = leg0_segments(b, ev)
        sin_all = np.abs(b.truth_state[np.concatenate([s[1] for s in segs]), 2])
        if len(segs) < 2 or min(len(s[1]) for s in segs) < 12 or sin_all.max() > 0.9:
            continue
        # every segment has consecutive rows in the generator (a clean crossing), and the segments follow each other
        if any(np.any(np.diff(s[2]) != 1) for s in segs) or any(segs[i + 1][2][0] - segs[i][2][-1] not in (0, 1, 2)
                                                                  for i in range(len(segs) - 1)):
            continue
        mine = np.nonzero(res.track_task // ns == ev)[0]
        heads = [i for i in range(len(m.merged_first)) if res.track_task[m.merged_first[i]] // ns == ev]
        leg0 = [i for i in heads if b.truth_leg[first_gid[m.merged_first[i]]] == 0]
        assert len(leg0) == 1, f"event {ev}: {len(leg0)} merged tracks on the outgoing leg"
        i = leg0[0]
        if segs[1][2][0] <= segs[0][2][-1]:
            continue  # the two sectors overlap in a row: G2 (rl_i < rf_j) does not link them by definition
        assert m.merged_nseg[i] == len(segs)
        assert m.merged_nhits[i] == sum(len(s[1]) for s in segs) == m.merged_nfit[i]
        chain, k = [], int(m.merged_first[i])
        while k >= 0:
            chain.append(k); k = int(m.next[k])
        for (sec, gids, _), k in zip(segs, chain):
            assert res.track_task[k] % ns == sec
            assert np.array_equal(res.track_hits(k), gids)
        g0 = segs[0][1][0]
        truth = b.truth_state[g0]
        assert m.merged_sector[i] == segs[0][0] and m.merged_x[i] == X[segs[0][2][0]]
        err = np.abs(m.merged_par[:, i] - truth) / np.maximum(np.abs(truth), [1.0, 1.0, 0.1, 0.1, 0.1])
        assert err.max() < 1e-5, (ev, err)
        n_by_seg[min(len(segs), 3)] += 1
    assert n_by_seg[2] >= 30 and n_by_seg[3] >= 3, n_by_seg
    assert len(mine) >= 1


def test_segments_of_different_tracks_are_never_linked():
    """36 well separated tracks per event that stay in their sector, and pairs of crossing tracks: a link only
    ever joins two segments of the SAME generated track."""
    rng = np.random.default_rng(12)
    evs = []
    for e in range(6):
        ph = (np.arange(18) + 0.5) * ALPHA + rng.uniform(-0.02, 0.02, 18)
        pt = rng.uniform(3.0, 8.0, 18)
        evs.append(generate_tracks_event(GEOM, pt, np.where(rng.random(18) < 0.5, -1.0, 1.0), ph,
                                         rng.uniform(-0.8, 0.8, 18), np.zeros(18), 0.1, 0.15, 0.0, rng, track_id_base=e * 100))
    for e in range(6):  # four crossing tracks per event, spread in z
        evs.append(generate_tracks_event(GEOM, rng.uniform(0.3, 0.8, 4), np.array([1.0, -1.0, 1.0, -1.0]),
                                         rng.uniform(0, 2 * np.pi, 4), np.array([-0.7, -0.25, 0.25, 0.7]), np.zeros(4),
                                         0.1, 0.15, 0.0, rng, track_id_base=1000 + e * 100))
    b = concat_batches(evs)
    prm = oracle.OracleParams()
    res = oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, params=prm)
    m = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, res, params=prm)
    first_gid = res.hit_cluster[res.track_hit_begin.astype(np.int64)]
    ns = b.geometry.n_sectors
    straight = res.track_task // ns < 6
    assert np.all(m.next[straight] == -1) and np.all(m.prev[straight] == -1)
    links = np.nonzero(m.next >= 0)[0]
    assert len(links) >= 6
    for i in links:
        j = int(m.next[i])
        assert b.truth_track[first_gid[i]] == b.truth_track[first_gid[j]] >= 0
        assert res.track_task[i] // ns == res.track_task[j] // ns and m.prev[j] == i


def _permuted(res, perm):
    beg = res.track_hit_begin.astype(np.int64)
    hits, begs = [], []
    for i in perm:
        begs.append(sum(len(h) for h in hits))
        hits.append(res.hit_cluster[beg[i]:beg[i] + int(res.track_nhits[i])])
    return types.SimpleNamespace(track_task=res.track_task[perm], track_hit_begin=np.array(begs, np.uint32),
                                 track_nhits=res.track_nhits[perm], track_x=res.track_x[perm],
                                 track_par=res.track_par[:, perm], track_cov=res.track_cov[:, perm],
                                 hit_cluster=np.concatenate(hits).astype(np.uint32))


def test_merge_does_not_depend_on_the_order_of_the_tracks():
    from tpc_workload import generate_config
    b = generate_config(1)
    prm = oracle.OracleParams(sigma_y=b.sigma_y, sigma_z=b.sigma_z)
    res = oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, params=prm)
    m0 = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, res, params=prm)
    assert m0.n_links > 300
    perm = np.random.default_rng(3).permutation(res.n_tracks)
    rp = _permuted(res, perm)
    m1 = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, rp, params=prm)
    fg0 = res.hit_cluster[res.track_hit_begin.astype(np.int64)]
    fg1 = rp.hit_cluster[rp.track_hit_begin.astype(np.int64)]
    links0 = {(int(fg0[i]), int(fg0[m0.next[i]])) for i in np.nonzero(m0.next >= 0)[0]}
    links1 = {(int(fg1[i]), int(fg1[m1.next[i]])) for i in np.nonzero(m1.next >= 0)[0]}
    assert links0 == links1
    by0 = {int(fg0[f]): k for k, f in enumerate(m0.merged_first)}
    for k1, f in enumerate(m1.merged_first):
        k0 = by0[int(fg1[f])]
        assert np.array_equal(m0.merged_par[:, k0], m1.merged_par[:, k1]) and m0.merged_nhits[k0] == m1.merged_nhits[k1]


def test_ties_go_to_the_smaller_first_hit_and_links_are_mutual():
    """G5, G6: two inner segments with the same outer end compete for one outer segment; the one whose first hit
    has the smaller gid gets it, the other gets nothing - whatever the order they are listed in."""
    rng = np.random.default_rng(13)
    while True:
        b = crossing_events(1, rng, 0.0, 0.0, pt_range=(0.4, 0.6))
        res = oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks)
        m = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, res)
        if m.n_links == 1 and res.n_tracks == 2:
            break
    a = int(np.nonzero(m.next >= 0)[0][0])
    bb = int(m.next[a])
    beg = res.track_hit_begin.astype(np.int64)
    ha, hb = res.track_hits(a), res.track_hits(bb)
    for order in ([0, 1, 2], [1, 0, 2], [2, 1, 0]):
        segs = [("A", ha, a), ("A2", ha[1:], a), ("B", hb, bb)]  # A2: same state, first hit dropped (larger first gid)
        segs = [segs[k] for k in order]
        hits = np.concatenate([s[1] for s in segs]).astype(np.uint32)
        begs = np.cumsum([0] + [len(s[1]) for s in segs[:-1]]).astype(np.uint32)
        src = [s[2] for s in segs]
        tr = types.SimpleNamespace(track_task=res.track_task[src], track_hit_begin=begs,
                                   track_nhits=np.array([len(s[1]) for s in segs], np.uint32), track_x=res.track_x[src],
                                   track_par=res.track_par[:, src], track_cov=res.track_cov[:, src], hit_cluster=hits)
        mm = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, tr)
        name = [s[0] for s in segs]
        iA, iA2, iB = name.index("A"), name.index("A2"), name.index("B")
        assert mm.n_links == 1 and mm.next[iA] == iB and mm.prev[iB] == iA and mm.next[iA2] == -1 and mm.prev[iA2] == -1


def _one_clean_crossing(seed):
    rng = np.random.default_rng(seed)
    while True:
        b = crossing_events(1, rng, 0.0, 0.0, pt_range=(0.4, 0.6))
        res = oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks)
        m = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, res)
        if m.n_links == 1 and res.n_tracks == 2:
            a = int(np.nonzero(m.next >= 0)[0][0])
            return b, res, a, int(m.next[a])


def _two_tracks(res, a, bb, hits_a, hits_b, par_b=None):
    src = [a, bb]
    par = res.track_par[:, src].copy()
    if par_b is not None:
        par[:, 1] = par_b
    return types.SimpleNamespace(track_task=res.track_task[src], track_hit_begin=np.array([0, len(hits_a)], np.uint32),
                                 track_nhits=np.array([len(hits_a), len(hits_b)], np.uint32), track_x=res.track_x[src],
                                 track_par=par, track_cov=res.track_cov[:, src],
                                 hit_cluster=np.concatenate([hits_a, hits_b]).astype(np.uint32))


def test_segments_that_share_a_row_are_not_linked():
    """G2: rl_i < rf_j, strictly.  The inner segment is given one more hit in the very row the outer one starts in
    (the merger reads only the row of a last hit): the pair must not be linked any more."""
    b, res, a, bb = _one_clean_crossing(21)
    ha, hb = res.track_hits(a), res.track_hits(bb)
    ok = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, _two_tracks(res, a, bb, ha, hb))
    assert ok.n_links == 1
    nr = b.geometry.n_rows
    row_of = lambda g: int((np.searchsorted(b.row_offsets, g, side="right") - 1) % nr)  # noqa: E731
    assert row_of(hb[0]) > row_of(ha[-1])
    # a cluster of the inner sector's own row rf_j would do; any gid of that ROW does, the row is all G2 reads
    same_row = np.concatenate([ha, hb[:1]])
    no = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, _two_tracks(res, a, bb, same_row, hb))
    assert no.n_links == 0 and no.next[0] == -1


def test_chi2_counts_all_five_parameters():
    """G4: an outer segment whose q/pT alone is off by ten standard deviations (of the two segments together; q/pT
    and its variance are not changed by ROTATE or TRANSPORT) adds 100 to chi2 and is not matched; off by one it is."""
    b, res, a, bb = _one_clean_crossing(22)
    ha, hb = res.track_hits(a), res.track_hits(bb)
    sig = np.sqrt(float(res.track_cov[14, a]) + float(res.track_cov[14, bb]))
    for n_sig, linked in ((1.0, 1), (10.0, 0)):
        par_b = res.track_par[:, bb].copy()
        par_b[4] += n_sig * sig
        m = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, _two_tracks(res, a, bb, ha, hb, par_b))
        assert m.n_links == linked, (n_sig, m.n_links)


def test_row_gap_and_chi2_cuts_decide_the_link():
    """G2, G4: the same pair is linked or not as merge_max_row_gap / merge_chi2_max say."""
    rng = np.random.default_rng(14)
    b = crossing_events(40, rng, 0.1, 0.15, pt_range=(0.4, 0.8))
    res = oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks)
    m = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, res)
    assert m.n_links >= 15
    nr = b.geometry.n_rows
    row_of = lambda g: (np.searchsorted(b.row_offsets, g, side="right") - 1) % nr  # noqa: E731
    beg = res.track_hit_begin.astype(np.int64)
    gaps = [int(row_of(res.hit_cluster[beg[m.next[i]]]) - row_of(res.hit_cluster[beg[i] + res.track_nhits[i] - 1]))
            for i in np.nonzero(m.next >= 0)[0]]
    assert min(gaps) >= 1 and max(gaps) <= 8
    for g in (1, 2, 4):
        mg = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, res, max_row_gap=g)
        assert mg.n_links == sum(1 for v in gaps if v <= g)
    assert oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, res, chi2_max=0.0).n_links == 0
    assert oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, res, chi2_max=1e9).n_links >= m.n_links


def test_merged_refit_has_unit_pulls():
    """Tracker + merger + refit on 3000 smeared single-track events that cross a sector boundary: (fit - truth)/sigma
    at the innermost hit has |mean| < 0.05 and width 1 +- 0.1 for all five parameters, <chi2/ndf> = 1 +- 0.03."""
    rng = np.random.default_rng(15)
    pulls, chi = [], []
    ns = GEOM.n_sectors
    while len(pulls) < 3000:
        b = crossing_events(1500, rng, 0.1, 0.15, pt_range=(0.3, 1.2))
        res = oracle.track(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, precision="f64")
        m = oracle.merge_refit(b.geometry, b.y, b.z, b.row_offsets, b.n_tasks, res, precision="f64")
        first_gid = res.hit_cluster[res.track_hit_begin.astype(np.int64)]
        for k in np.nonzero((m.merged_nseg >= 2) & (m.merged_nfit == m.merged_nhits) & (m.merged_nhits >= 40))[0]:
            g0 = first_gid[m.merged_first[k]]
            if b.truth_leg[g0] != 0:
                continue
            ev = res.track_task[m.merged_first[k]] // ns
            segs = leg0_segments(b, ev)
            if np.abs(b.truth_state[np.concatenate([s_[1] for s_ in segs]), 2]).max() > 0.85:
                continue
            assert m.merged_ndf[k] == 2 * m.merged_nfit[k] - 5
            truth = b.truth_state[g0]
            pulls.append((m.merged_par[:, k] - truth) / np.sqrt(m.merged_cov[[0, 2, 5, 9, 14], k]))
            chi.append(m.merged_chi2[k] / m.merged_ndf[k])
    pulls = np.array(pulls)
    assert np.all(np.abs(pulls.mean(axis=0)) < 0.05), pulls.mean(axis=0)
    assert np.all(np.abs(pulls.std(axis=0) - 1.0) < 0.1), pulls.std(axis=0)
    assert abs(np.mean(chi) - 1.0) < 0.03, np.mean(chi)


def test_straight_line_across_a_boundary_equals_least_squares_in_global_coordinates():
    """Bz = 0, hits in two sectors: the refit (rotation at the boundary included) must give the weighted
    least-squares line, solved here by Gauss-Newton on the residuals along each sector's own y axis and z.
    The refit starts from the truth with a wide covariance and linearises where Gauss-Newton iterates, so it sits
    within a tenth of a sigma of the least-squares solution; a wrong sign or a transposed rotation moves it by
    many sigma."""
    import dataclasses
    g0 = dataclasses.replace(GEOM, bz_kgauss=0.0)
    rng = np.random.default_rng(16)
    sy, sz = 0.1, 0.15
    done = 0
    for trial in range(400):
        kA = int(rng.integers(0, 18))
        d = 1 if rng.random() < 0.5 else -1
        kB = (kA + d) % 18
        # a line through the boundary between sectors kA and kB at radius ~ 160 cm
        al_edge = sector_angle(kA) + d * ALPHA / 2
        r_edge = rng.uniform(130, 200)
        psi = al_edge + d * rng.uniform(0.15, 0.5)     # heading towards kB
        P0 = np.array([r_edge * np.cos(al_edge), r_edge * np.sin(al_edge)])
        u = np.array([np.cos(psi), np.sin(psi)])
        tz, z0 = rng.uniform(-0.5, 0.5), rng.uniform(20, 200)

        def hits_in(k):
            al = sector_angle(k)
            ex, ey = np.array([np.cos(al), np.sin(al)]), np.array([-np.sin(al), np.cos(al)])
            out = []
            for r in range(GEOM.n_rows):
                lam = (X[r] - P0 @ ex) / (u @ ex)
                P = P0 + lam * u
                yl = P @ ey
                if abs(yl) <= X[r] * np.tan(np.deg2rad(10.0)) and ((k == kA and lam < 0) or (k == kB and lam > 0)):
                    out.append((k, r, yl, z0 + tz * lam, lam))
            return out
        hA, hB = hits_in(kA), hits_in(kB)
        if len(hA) < 12 or len(hB) < 12:
            continue
        hits = sorted(hA + hB, key=lambda h: -h[4])            # outermost first
        sec = np.array([h[0] for h in hits]); row = np.array([h[1] for h in hits])
        ym = np.array([h[2] for h in hits]) + sy * rng.standard_normal(len(hits))
        zm = np.array([h[3] for h in hits]) + sz * rng.standard_normal(len(hits))
        lam = np.array([h[4] for h in hits])
        # Gauss-Newton for the global line (point Q on the normal through P0, heading angle, z at lam = 0, slope)
        def resid(par):
            off, ang, zz, tt = par
            uu = np.array([np.cos(ang), np.sin(ang)]); nn = np.array([-uu[1], uu[0]])
            Q = P0 + off * nn
            out = []
            for k_, r_, y_, z_ in zip(sec, row, ym, zm):
                al = sector_angle(k_)
                ex, ey = np.array([np.cos(al), np.sin(al)]), np.array([-np.sin(al), np.cos(al)])
                l_ = (X[r_] - Q @ ex) / (uu @ ex)
                out += [((Q + l_ * uu) @ ey - y_) / sy, (zz + tt * l_ - z_) / sz]
            return np.array(out)
        par = np.array([0.0, psi, z0, tz])
        for _ in range(6):
            r0 = resid(par)
            J = np.array([(resid(par + dv) - r0) / 1e-6 for dv in 1e-6 * np.eye(4)]).T
            par = par - np.linalg.solve(J.T @ J, J.T @ r0)
        cov = np.linalg.inv(J.T @ J)
        # the least-squares line at the innermost hit, in its sector's frame
        k_in, r_in = int(sec[-1]), int(row[-1])
        al = sector_angle(k_in)
        ex, ey = np.array([np.cos(al), np.sin(al)]), np.array([-np.sin(al), np.cos(al)])
        uu = np.array([np.cos(par[1]), np.sin(par[1])]); Q = P0 + par[0] * np.array([-uu[1], uu[0]])
        l_in = (X[r_in] - Q @ ex) / (uu @ ex)
        ref = np.array([(Q + l_in * uu) @ ey, par[2] + par[3] * l_in, np.sin(par[1] - al), par[3]])
        # start state: the truth at the outermost hit with a generous covariance (F1 multiplies it by 100)
        k_out, r_out = int(sec[0]), int(row[0])
        alo = sector_angle(k_out)
        p_start = np.array([hits[0][2], hits[0][3], np.sin(psi - alo), tz, 0.0])
        c_start = pack_cov(np.diag([sy**2, sz**2, 1e-4, 1e-4, 1e-6]))
        n_fit, x, p, c, chi2, ndf, sector = oracle.refit_hits(g0, sec, row, ym, zm, X[r_out], p_start, c_start, k_out)
        assert n_fit == len(hits) and sector == k_in and x == X[r_in]
        sig = np.sqrt(np.diag(unpack_cov(c))[:4])
        assert np.all(np.abs(p[:4] - ref) < 0.1 * sig), (trial, (p[:4] - ref) / sig)
        done += 1
        if done == 40:
            break
    assert done == 40
