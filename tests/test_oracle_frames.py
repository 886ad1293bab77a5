"""Pins of SPEC 11 (time-frame mode: "slice the time frames along the time / beam axis, process
the slices individually, and merge the track segments afterwards") on the CPU oracle."""
from __future__ import annotations

import dataclasses

import numpy as np

import oracle
from tpc_workload import default_geometry, generate_event, generate_tracks_event, make_frame, CONFIGS

GEOM = default_geometry()
X = GEOM.row_x.astype(np.float64)


def test_without_projection_the_tracker_does_not_care_where_z_starts():
    """nf_z_projection = 0: an event shifted by 300 cm along z (each side away from the centre, as in a frame) gives
    the same links, the same tracks hit for hit, and the same parameters with z moved by the shift (fp64)."""
    ev = generate_event(GEOM, dataclasses.replace(CONFIGS[1]["spec"], n_primaries=300), 5)
    ns, nr = GEOM.n_sectors, GEOM.n_rows
    sec = np.repeat(np.arange(ns * nr), np.diff(ev.row_offsets.astype(np.int64))) // nr
    sgn = np.where(2 * sec < ns, 1.0, -1.0)
    big = dataclasses.replace(GEOM, z_max=600.0)
    prm = oracle.OracleParams(nf_z_projection=0, nf_hz=2.5)
    y, z = ev.y.astype(np.float64), ev.z.astype(np.float64)
    a = oracle.track(big, y, z, ev.row_offsets, ev.n_tasks, params=prm, precision="f64")
    b = oracle.track(big, y, z + 300.0 * sgn, ev.row_offsets, ev.n_tasks, params=prm, precision="f64")
    assert a.n_tracks > 300
    assert np.array_equal(a.link_up, b.link_up) and np.array_equal(a.link_dn, b.link_dn)
    assert np.array_equal(a.hit_cluster, b.hit_cluster) and np.array_equal(a.track_nhits, b.track_nhits)
    dz = 300.0 * np.where(2 * (a.track_task % ns) < ns, 1.0, -1.0)
    assert np.allclose(b.track_par[1] - dz, a.track_par[1], atol=1e-9, rtol=0)
    for k in (0, 2, 3, 4):
        assert np.allclose(b.track_par[k], a.track_par[k], atol=1e-9, rtol=1e-9)
    # and WITH the projection of N1 the shifted event loses a good part of its links (the inner rows, where X[r+1]/X[r] - 1 is largest): that is why the switch exists
    c = oracle.track(big, y, z + 300.0 * sgn, ev.row_offsets, ev.n_tasks, params=oracle.OracleParams(nf_hz=2.5),
                     precision="f64")
    assert (c.link_up >= 0).sum() < 0.8 * (a.link_up >= 0).sum()


def _single_track_frame(rng, n, sigma_y, sigma_z, slice_len=250.0, n_slices=3):
    """n single-track events, each shifted so that its outgoing leg crosses the first slice boundary mid-way."""
    evs, shifts = [], []
    while len(evs) < n:
        pt = np.exp(rng.uniform(np.log(0.4), np.log(3.0), 1))
        eta = rng.choice([-1.0, 1.0]) * rng.uniform(0.3, 0.9, 1)
        ev = generate_tracks_event(GEOM, pt, np.where(rng.random(1) < 0.5, -1.0, 1.0), rng.uniform(0, 2 * np.pi, 1), eta,
                                   np.zeros(1), sigma_y, sigma_z, 0.0, rng, track_id_base=0)
        leg0 = ev.truth_leg == 0
        if leg0.sum() < 80:
            continue
        zz = np.abs(ev.truth_state[leg0, 1])
        z_mid = float(np.median(zz))
        evs.append(ev)
        shifts.append(slice_len - z_mid + rng.uniform(-20, 20))
    return evs, shifts


def test_noiseless_tracks_across_a_slice_boundary_are_merged_and_refitted_to_truth():
    """Every event is a frame of its own (frame index = event): its one track crosses from slice 0 into slice 1 (and
    often into a neighbouring sector as well); the merged track holds every cluster of the outgoing leg and its
    refit equals truth to 1e-5 (fp64 instantiation, exact fp64 crossings as input)."""
    rng = np.random.default_rng(31)
    evs, shifts = _single_track_frame(rng, 60, 0.0, 0.0)
    prm = oracle.OracleParams(nf_z_projection=0, nf_hz=2.5)
    ns, nr, n_sl = GEOM.n_sectors, GEOM.n_rows, 3
    n_checked = n_two_kinds = 0
    for ev, sh in zip(evs, shifts):
        fr = make_frame([ev], [sh], 250.0, n_sl, seed=1)
        y64, z64 = fr.truth_state[:, 0].copy(), fr.truth_state[:, 1].copy()
        res = oracle.track(fr.geometry, y64, z64, fr.row_offsets, fr.n_tasks, params=prm, precision="f64")
        m = oracle.merge_refit(fr.geometry, y64, z64, fr.row_offsets, fr.n_tasks, res, params=prm, precision="f64",
                               n_slices=n_sl)
        tr = np.searchsorted(fr.row_offsets, np.arange(fr.n_clusters), side="right") - 1
        leg0 = np.nonzero(fr.truth_leg == 0)[0]
        if np.abs(fr.truth_state[leg0, 2]).max() > 0.9:
            continue
        # the (slice, sector) pieces of the leg, in row order; need clean pieces of >= 12 consecutive rows
        task0, row0 = tr[leg0] // nr, tr[leg0] % nr
        order = np.argsort(row0, kind="stable")
        pieces, cur = [], [leg0[order[0]]]
        for a, b in zip(order[:-1], order[1:]):
            if task0[a] == task0[b]:
                cur.append(leg0[b])
            else:
                pieces.append(cur); cur = [leg0[b]]
        pieces.append(cur)
        rows_ok = all(len(p) >= 12 for p in pieces) and len(np.unique(row0)) == len(row0)
        if len(pieces) < 2 or not rows_ok:
            continue
        first_gid = res.hit_cluster[res.track_hit_begin.astype(np.int64)]
        mine = [k for k in range(len(m.merged_first)) if fr.truth_leg[first_gid[m.merged_first[k]]] == 0]
        assert len(mine) == 1, (len(pieces), len(mine))
        k = mine[0]
        assert m.merged_nseg[k] == len(pieces) and m.merged_nhits[k] == len(leg0) == m.merged_nfit[k]
        kinds = set()
        i = int(m.merged_first[k])
        while m.next[i] >= 0:
            j = int(m.next[i])
            ti, tj = int(res.track_task[i]), int(res.track_task[j])
            kinds.add("slice" if ti % ns == tj % ns else "sector")
            assert (ti % ns == tj % ns and abs(ti // ns - tj // ns) == 1) or (ti // ns == tj // ns and ti % ns != tj % ns)
            i = j
        g0 = pieces[0][0]
        truth = fr.truth_state[g0]
        err = np.abs(m.merged_par[:, k] - truth) / np.maximum(np.abs(truth), [1.0, 1.0, 0.1, 0.1, 0.1])
        assert err.max() < 1e-5, err
        n_checked += 1
        n_two_kinds += len(kinds) == 2
        assert "slice" in kinds
    assert n_checked >= 25 and n_two_kinds >= 3, (n_checked, n_two_kinds)


def test_frame_of_overlapping_events_links_only_neighbours_and_the_same_track():
    """Six peripheral events overlaid at random shifts, four slices: every link joins either neighbouring sectors of
    one slice or one sector of neighbouring slices; at least 99 % of the links join two segments of the same
    generated track; frame tracking finds about as many merged tracks as tracking the events one by one."""
    spec = CONFIGS[1]["spec"]
    evs = [generate_event(GEOM, spec, 300 + i) for i in range(6)]
    shifts = np.sort(np.random.default_rng(2).uniform(0, 750, 6))
    fr = make_frame(evs, shifts, 250.0, 4, seed=9)
    prm = oracle.OracleParams(sigma_y=fr.sigma_y, sigma_z=fr.sigma_z, nf_z_projection=0, nf_hz=2.5)
    res = oracle.track(fr.geometry, fr.y, fr.z, fr.row_offsets, fr.n_tasks, params=prm)
    m = oracle.merge_refit(fr.geometry, fr.y, fr.z, fr.row_offsets, fr.n_tasks, res, params=prm, n_slices=4)
    ns = GEOM.n_sectors
    first_gid = res.hit_cluster[res.track_hit_begin.astype(np.int64)]
    links = np.nonzero(m.next >= 0)[0]
    assert len(links) > 2000
    same = 0
    n_slice_links = 0
    for i in links:
        j = int(m.next[i])
        ti, tj = int(res.track_task[i]), int(res.track_task[j])
        si, sj, li, lj = ti % ns, tj % ns, ti // ns, tj // ns
        if li == lj:
            assert si // 18 == sj // 18 and (si % 18 - sj % 18) % 18 in (1, 17)
        else:
            assert si == sj and abs(li - lj) == 1
            n_slice_links += 1
        same += fr.truth_track[first_gid[i]] == fr.truth_track[first_gid[j]] >= 0
    assert n_slice_links > 200
    assert same >= 0.99 * len(links), (same, len(links))
    alone = 0
    for e in evs:
        p1 = oracle.OracleParams(sigma_y=e.sigma_y, sigma_z=e.sigma_z)
        r = oracle.track(GEOM, e.y, e.z, e.row_offsets, e.n_tasks, params=p1)
        alone += len(oracle.merge_refit(GEOM, e.y, e.z, e.row_offsets, e.n_tasks, r, params=p1).merged_first)
    assert abs(len(m.merged_first) - alone) < 0.08 * alone, (len(m.merged_first), alone)
    # n_slices = 1 on the same tracks: no link may cross a slice, so there are fewer
    m1 = oracle.merge_refit(fr.geometry, fr.y, fr.z, fr.row_offsets, fr.n_tasks, res, params=prm, n_slices=1)
    assert m1.n_links < m.n_links


def test_slicer_hand_built_and_properties():
    """SLICE: a hand-built frame (2 sectors, 3 rows, slices of 100 cm) and the properties on a generated one."""
    from oracle.frames import slice_frames
    # sector 0 row 0: zeta 10, 250, 99.9, 100 ; sector 0 row 2: 5 ; sector 1 row 1: -120, -20, -350 (C-side sign)
    y = np.arange(8, dtype=np.float32)
    z = np.array([10, 250, 99.9, 100, 5, -120, -20, -350], np.float32)
    ro = np.array([0, 4, 4, 5, 5, 8, 8], np.uint32)
    yo, zo, src, ro_out = slice_frames(y, z, ro, 2, 2, 3, 100.0, 3)
    # slices: 0,2,0,1 | 0 | 1,0,2(clipped from 3)   -> output order (slice, sector, row, input order)
    assert src.tolist() == [0, 2, 4, 6, 3, 5, 1, 7]
    assert np.array_equal(yo, y[src]) and np.array_equal(zo, z[src])
    want_counts = {(0, 0, 0): 2, (0, 0, 2): 1, (0, 1, 1): 1, (1, 0, 0): 1, (1, 1, 1): 1, (2, 0, 0): 1, (2, 1, 1): 1}
    for sl in range(3):
        for sec in range(2):
            for r in range(3):
                k = (sl * 2 + sec) * 3 + r
                assert ro_out[k + 1] - ro_out[k] == want_counts.get((sl, sec, r), 0)
    # a generated frame: permutation, stability inside a row, every cluster in the slice of its zeta
    spec = CONFIGS[1]["spec"]
    evs = [generate_event(GEOM, spec, 500 + i) for i in range(3)]
    fr = make_frame(evs, [0.0, 200.0, 420.0], 1000.0, 1, seed=3)           # one slice = not yet sliced
    yo, zo, src, ro_out = slice_frames(fr.y, fr.z, fr.row_offsets, 36, 36, 159, 250.0, 4)
    assert np.array_equal(np.sort(src), np.arange(fr.n_clusters))
    tr_out = np.repeat(np.arange(len(ro_out) - 1), np.diff(ro_out.astype(np.int64)))
    sl = tr_out // 159 // 36
    assert np.all(sl == np.minimum((np.abs(zo) * (np.float32(1) / np.float32(250.0))).astype(np.int64), 3))
    same_row = tr_out[1:] == tr_out[:-1]
    assert np.all(src[1:][same_row] > src[:-1][same_row])
