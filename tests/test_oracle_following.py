"""Pins of the FOLLOWING half of the oracle (docs/ARITH_SPEC.md 5.3 H1-H6, 6 K2-K7) - CPU only.

Every expectation here is worked out by hand (or with textbook regression / matrix-form Kalman algebra in
numpy) from the SPEC, never by re-typing the oracle's sequence:

* hand-built straight tracks at Bz = 0 on the line y = 0, z = const.  Every residual of such a track is exactly
  zero, so the fitted state stays exactly on the line (U5 adds k_j*0) and the prediction in every row is exactly
  (0, z): the distance of a planted cluster to the prediction is known exactly.
* the metric of H5 is dy^2*ez + dz^2*ey, i.e. (up to the common factor ey*ez) dy^2/ey + dz^2/ez.  For the line above
  the y and z regressions have the same design (f02 = f13 = dx), so ey : ez = sigma_y^2 : sigma_z^2 = 1 : 2.25 up to
  the 1e-4 weight of the seed prior.
* the covariance of the prediction is that of the weighted linear regression over the hits fitted so far:
  var(y_pred) = sigma_y^2 * (1/n + (x - xbar)^2 / Sxx), which fixes the 4-sigma window of H2 independently.

tests/mutants.md lists the plausible mistakes these tests were built to kill (tests/mutation_check.py re-runs them).
"""
import dataclasses

import numpy as np
import pytest

import oracle
from oracle import OracleParams
from helpers import A_PER_KG, batch_from_rows, pack_cov, unpack_cov, single_track_events
from tpc_workload import default_geometry

G0 = dataclasses.replace(default_geometry(n_sectors=1), bz_kgauss=0.0)  # straight lines
SY, SZ = 0.1, 0.15
Z0 = 10.0


def run(b, g=G0, **kw):
    return oracle.track(g, b.y, b.z, b.row_offsets, b.n_tasks, dump_tracklets=True, **kw)


def line_rows(rows, z=Z0):
    return {(0, r): [(0.0, z)] for r in rows}


def gid_table(pts, n_rows=159):
    """{(row, k): gid} for batch_from_rows' order (task 0)."""
    out, g = {}, 0
    for r in range(n_rows):
        for k in range(len(pts.get((0, r), []))):
            out[(r, k)] = g
            g += 1
    return out


def tracklet_from(res, start_gid):
    i = np.nonzero(res.tracklet_start == start_gid)[0]
    assert len(i) == 1, f"no tracklet starts at gid {start_gid}"
    return res.tracklet_map[int(i[0])]


def pred_var(rows_fitted, row, sigma2, g=G0):
    """Variance of the straight-line regression over rows_fitted, evaluated at `row` (diffuse prior)."""
    x = g.row_x[list(rows_fitted)].astype(np.float64)
    xb = x.mean()
    return sigma2 * (1.0 / len(x) + (float(g.row_x[row]) - xb) ** 2 / ((x - xb) ** 2).sum())


# A line with hits in rows 20..30: the clusters of rows 20 and 30 have only one neighbour row (pair or nothing,
# R5), so the CA chain is rows 21..29 (start hit in row 21); row 30 is found by the up pass, row 20 by the down pass.
BASE_ROWS = list(range(20, 31))
# Hits that carry information when the up pass reaches row 32 (row 31 is left empty): K1 takes the start hit (row 21)
# only as the linearisation point of the slope (prior variance c0_sinphi = 1 = diffuse) - the covariance starts as
# sigma^2 at the row-22 hit - so the fit is the regression over rows 22..30.
FITTED_AT_32 = list(range(22, 31))


# ------------------------------------------------------------------------------------------- SEARCH (H1-H6)
def test_search_metric_weights_dy2_by_ez_and_dz2_by_ey():
    """H5.  Three candidates in row 32 at (dy, dz) = A (0.11, 0), B (0, 0.125), C (0.075, 0.075); with
    1/ey : 1/ez = 2.25 : 1 the normalised distances are
        H5 (dy^2*2.25 + dz^2)      A .0272  B .0156  C .0183  -> B
        weights swapped            A .0121  B .0352  C .0183  -> A
        plain Euclid               A .0121  B .0156  C .0113  -> C
    so each of the three metrics picks a different cluster."""
    for order in ([0, 1, 2], [2, 1, 0], [1, 2, 0]):
        cand = [(0.11, Z0), (0.0, Z0 + 0.125), (0.075, Z0 + 0.075)]
        pts = line_rows(BASE_ROWS)
        pts[(0, 32)] = [cand[k] for k in order]
        gids = gid_table(pts)
        res = run(batch_from_rows(G0, pts))
        m = tracklet_from(res, gids[(21, 0)])
        assert m[32] == gids[(32, order.index(1))], "H5 must pick B = (0, +0.125)"
        assert m[31] == -1 and (m[20:31] >= 0).all()


@pytest.mark.parametrize("bins", [(2.0, 2.0), (1.0, 1.0), (2.0, 20.0)])
def test_search_tie_goes_to_smaller_gid(bins):
    """H6.  Exact duplicates, and two clusters at dz = -/+0.0625 (equal distance, different z bins at bin size 2:
    (10.9375+1)/2 = 5.97, (11.0625+1)/2 = 6.03, so the grid visits the -0.0625 one first): the smaller gid wins
    whatever the visiting order."""
    prm = OracleParams(grid_bin_min=bins[0], grid_bin_max=bins[1])
    z = 11.0
    for cand in ([(0.3, z), (0.0625, z), (0.0625, z)], [(0.0625, z), (0.3, z), (0.0625, z)],
                 [(0.0, z - 0.0625), (0.0, z + 0.0625)], [(0.0, z + 0.0625), (0.0, z - 0.0625)],
                 [(-0.0625, z), (0.0625, z)], [(0.0625, z), (-0.0625, z)]):
        pts = line_rows(BASE_ROWS, z)
        pts[(0, 32)] = cand
        gids = gid_table(pts)
        res = run(batch_from_rows(G0, pts), params=prm)
        m = tracklet_from(res, gids[(21, 0)])
        near = [k for k, (y, zz) in enumerate(cand) if abs(y) + abs(zz - z) < 0.1]
        assert len(near) == 2
        assert m[32] == gids[(32, min(near))], (cand, int(m[32]))


def test_search_window_cap_and_boundaries():
    """H2/H4.  With accept_k2 = 1e6 the cap decides: hy2 = hz2 = search_max^2 = 9, boundary inclusive."""
    prm = OracleParams(accept_k2=1e6)
    up = lambda v: float(np.nextafter(np.float32(v), np.float32(1e9)))  # noqa: E731
    cases = [((3.0, Z0), True),                 # dy^2 == hy2 exactly: valid (H4 is <=)
             ((up(3.0), Z0), False),             # one ulp outside
             ((-3.0, Z0), True),
             ((0.0, Z0 + 3.0), True),            # dz^2 == hz2 exactly (13.0 - 10.0 is exact)
             ((0.0, up(Z0 + 3.0)), False),       # (13.000001 - 10)^2 > 9
             ((0.0, Z0 - 2.5), True),            # well inside in z: kills a halved z window
             ((2.5, Z0 + 2.5), True),            # the window is a box, not an ellipse
             ((3.5, Z0), False), ((0.0, Z0 + 3.5), False)]
    for c, valid in cases:
        pts = line_rows(BASE_ROWS)
        pts[(0, 32)] = [c]
        gids = gid_table(pts)
        m = tracklet_from(run(batch_from_rows(G0, pts), params=prm), gids[(21, 0)])
        assert (m[32] == gids[(32, 0)]) == valid, (c, valid)
        assert (m[32] == -1) == (not valid)


def test_search_window_is_k2_sigma_when_below_the_cap():
    """H1/H2 with the defaults (K2 = 16 -> 4 sigma, far below the 3 cm cap).  ey = var(y_pred) + sigma_y^2 from the
    regression over the nine rows 22..30 that carry weight (see FITTED_AT_32), evaluated at row 32."""
    ey = pred_var(FITTED_AT_32, 32, SY ** 2) + SY ** 2
    ez = pred_var(FITTED_AT_32, 32, SZ ** 2) + SZ ** 2
    by, bz = 4.0 * np.sqrt(ey), 4.0 * np.sqrt(ez)
    assert 0.4 < by < 0.8 and 0.6 < bz < 1.2  # the construction: both well under the cap of 3 cm
    cases = [((0.97 * by, Z0), True), ((1.03 * by, Z0), False), ((-0.97 * by, Z0), True),
             ((0.0, Z0 + 0.97 * bz), True), ((0.0, Z0 + 1.03 * bz), False), ((0.0, Z0 - 1.03 * bz), False),
             ((0.97 * by, Z0 - 0.97 * bz), True),  # box: both inside
             ((1.0, Z0), False),                   # inside the cap, outside 4 sigma: the MIN of H2 decides
             ((0.0, Z0 + 1.4), False)]
    for c, valid in cases:
        pts = line_rows(BASE_ROWS)
        pts[(0, 32)] = [c]
        gids = gid_table(pts)
        m = tracklet_from(run(batch_from_rows(G0, pts)), gids[(21, 0)])
        assert (m[32] == gids[(32, 0)]) == valid, (c, valid)
    # the y window uses ey and the z window ez (not the other way round): 0.97*bz in y is outside, since bz > by
    assert 0.97 * bz > 1.03 * by
    pts = line_rows(BASE_ROWS)
    pts[(0, 32)] = [(0.97 * bz, Z0)]
    gids = gid_table(pts)
    assert tracklet_from(run(batch_from_rows(G0, pts)), gids[(21, 0)])[32] == -1


# ------------------------------------------------------------------------------------------- gaps (K3, K5)
def test_up_pass_gap_logic():
    """K3.  Hits in rows 20-30, [31-34 missing], 35, 36, [37-40 missing], 41, [42-46 missing], 47-60.
    max_row_gap = 4: a gap of 4 is bridged and the count restarts after a hit (two gaps of 4 do not add up); the gap
    of 5 ends the pass, lastRow = 41.  The second line piece (47-60) is its own tracklet: its down pass crosses 46..42
    (five misses below its firstRow) and stops before it reaches row 41."""
    rows = list(range(20, 31)) + [35, 36, 41] + list(range(47, 61))
    pts = line_rows(rows)
    gids = gid_table(pts)
    res = run(batch_from_rows(G0, pts))
    m = tracklet_from(res, gids[(21, 0)])
    want = np.full(159, -1)
    for r in list(range(20, 31)) + [35, 36, 41]:
        want[r] = gids[(r, 0)]
    np.testing.assert_array_equal(m, want)
    m2 = tracklet_from(res, gids[(48, 0)])
    want2 = np.full(159, -1)
    for r in range(47, 61):
        want2[r] = gids[(r, 0)]
    np.testing.assert_array_equal(m2, want2)
    # with max_row_gap = 5 the first tracklet runs through to row 60, with 3 it ends at row 30
    m5 = tracklet_from(run(batch_from_rows(G0, pts), params=OracleParams(max_row_gap=5)), gids[(21, 0)])
    assert set(np.nonzero(m5 >= 0)[0]) == set(rows)
    m3 = tracklet_from(run(batch_from_rows(G0, pts), params=OracleParams(max_row_gap=3)), gids[(21, 0)])
    assert set(np.nonzero(m3 >= 0)[0]) == set(range(20, 31))
    # max_row_gap = 0: the first miss ends a pass
    pts0 = line_rows(list(range(20, 31)) + [32])
    m0 = tracklet_from(run(batch_from_rows(G0, pts0), params=OracleParams(max_row_gap=0)), gid_table(pts0)[(21, 0)])
    assert set(np.nonzero(m0 >= 0)[0]) == set(range(20, 31))


def _line_fit_cov(rows, s2, g=G0, C=None, x=None):
    """Textbook Kalman filter of a straight line, state (y, dy/dx): covariance after fitting `rows` in the order
    given, starting either from K1's seed (sigma^2 at rows[0], slope prior 1) or from (C, x)."""
    X = g.row_x.astype(np.float64)
    if C is None:
        C, x, rows = np.diag([s2, 1.0]), X[rows[0]], rows[1:]
    for r in rows:
        F = np.array([[1.0, X[r] - x], [0.0, 1.0]])
        C, x = F @ C @ F.T, X[r]
        K = C[:, :1] / (C[0, 0] + s2)
        C = C - K @ C[:1, :]
    return C, x


def test_down_pass_gap_logic_and_in_span_search():
    """K5, with turn_cov_scale = 1e4 so that the down pass starts from an (almost) flat prior.
    Line hits in rows 20-30, 32, 33; row 31 holds a cluster 0.72 cm off in y.
    Up pass at row 31: window 4*sqrt(var_pred + sigma_y^2) = 0.49 cm (fit over rows 22..30) -> miss; rows 32, 33 are
    found, then five misses end the pass, lastRow = 33.  The down pass reaches row 31 with only the hits of rows 33
    and 32 behind its flat prior: var_pred ~ sigma_y^2 (2^2 + 1^2), window 0.95 cm -> the 0.72 cm cluster is picked
    up INSIDE the span (a miss there would not have counted towards a gap either).
    Below firstRow = 20: rows 19, 18 missing, 17 hit, 16-14 missing, 13 hit (gaps of 2 and 3 do not add up: the count
    restarts at a hit), 12-8 missing = 5 misses -> stop; the cluster in row 7 is never reached."""
    X = G0.row_x.astype(np.float64)
    C, x = _line_fit_cov(list(range(22, 31)), SY ** 2)
    up_win = 4.0 * np.sqrt(C[0, 0] + 2 * (X[31] - x) * C[0, 1] + (X[31] - x) ** 2 * C[1, 1] + SY ** 2)
    C, x = _line_fit_cov([32, 33], SY ** 2, C=C, x=x)
    C, x = _line_fit_cov([33, 32], SY ** 2, C=C * 1e4, x=x)
    dn_win = 4.0 * np.sqrt(C[0, 0] + 2 * (X[31] - x) * C[0, 1] + (X[31] - x) ** 2 * C[1, 1] + SY ** 2)
    assert up_win < 0.55 < 0.72 < 0.90 < dn_win  # the construction
    prm = OracleParams(turn_cov_scale=1e4)
    rows = [7, 13, 17] + list(range(20, 31)) + [32, 33]
    pts = line_rows(rows)
    pts[(0, 31)] = [(0.72, Z0)]
    gids = gid_table(pts)
    res = run(batch_from_rows(G0, pts), params=prm)
    m = tracklet_from(res, gids[(21, 0)])
    want = np.full(159, -1)
    for r in [13, 17] + list(range(20, 34)):
        want[r] = gids[(r, 0)]
    np.testing.assert_array_equal(m, want)
    # in-span misses do not count towards the gap below firstRow: rows 31-34 missing (bridged by the up pass),
    # then two missing rows below firstRow and a hit in row 17 - 4 + 2 misses in total, but only 2 count
    rows = [17] + list(range(20, 31)) + list(range(35, 45))
    pts = line_rows(rows)
    gids = gid_table(pts)
    m = tracklet_from(run(batch_from_rows(G0, pts)), gids[(21, 0)])
    assert set(np.nonzero(m >= 0)[0]) == set(rows)


# ------------------------------------------------------------------------------------------- K2 failure, P4
def test_transport_fails_when_current_sinphi_is_beyond_the_limit():
    """P4 (D2): the test is on |s| AND |s1|.  s = 0.96 bending back to s1 = 0.90 must still fail."""
    a = A_PER_KG * 5.0
    p = np.array([0.0, 0.0, 0.96, 0.0, 10.0])  # k = a*q < 0: sinphi falls with x
    c = pack_cov(np.eye(5))
    s1 = 0.96 + a * 10.0 * 4.0
    assert 0.85 < s1 < 0.95
    for prec in ("f64", "f32"):
        ok, x1, p1, c1 = oracle.transport(100.0, p, c, 104.0, a, precision=prec)
        assert not ok and x1 == 100.0
        np.testing.assert_array_equal(p1, p.astype(p1.dtype))
    ok, *_ = oracle.transport(100.0, np.array([0.0, 0.0, 0.94, 0.0, 10.0]), c, 104.0, a)
    assert ok


def test_chain_fit_stops_where_sinphi_passes_the_limit():
    """K2 -> K4.  A noiseless pT = 0.15 GeV helix (R = 100 cm) whose sin(phi) in the sector frame grows through
    0.95 inside the CA chain: the chain hits beyond the row where the transport fails are NOT in the tracklet
    although they are linked, and nothing above that row is picked up.  (Continuing into the up pass after a K2
    failure is not a different reading: the up pass would start with the very transport that just failed.)"""
    g = default_geometry(n_sectors=1)
    a = A_PER_KG * 5.0
    q = -10.0 / 1.5  # 1/pT = 6.67 c/GeV, k = a*q > 0
    k = a * q
    x0, s0 = float(g.row_x[30]), 0.55
    # circle through (x0, 0) with direction sin(phi) = s0: sin(phi)(x) = s0 + k (x - x0); y from the closed form
    rows = list(range(30, 75))
    xs = g.row_x[rows].astype(np.float64)
    s = s0 + k * (xs - x0)
    keep = np.abs(s) < 0.995
    rows, xs, s = [r for r, kk in zip(rows, keep) if kk], xs[keep], s[keep]
    y = (np.sqrt(1 - s0 ** 2) - np.sqrt(1 - s ** 2)) / k
    phi = np.arcsin(s)
    z = 20.0 + 0.3 * (phi - np.arcsin(s0)) / k
    assert s.max() > 0.97
    pts = {(0, r): [(float(yy), float(zz))] for r, yy, zz in zip(rows, y, z)}
    b = batch_from_rows(g, pts)
    # the default neighbour window (2 cm in y per row) cannot link beyond sin(phi) ~ 0.89 (dy/dx = tan(phi) > 2):
    # open it so that the CA chain really runs through the limit
    prm = OracleParams(nf_hy=12.0, nf_hz=5.0, nf_chi2_max=1e6)
    res = oracle.track(g, b.y.astype(np.float64), b.z.astype(np.float64), b.row_offsets, 1, precision="f64",
                       dump_tracklets=True, params=prm)
    gids = gid_table(pts)
    # the chain really runs past the limit (the CA does not know about sin(phi))
    linked = [r for r in rows if res.clean_up[gids[(r, 0)]] >= 0]
    s_of = dict(zip(rows, s))
    assert max(s_of[r] for r in linked) > 0.96
    m = tracklet_from(res, gids[(rows[1], 0)])
    got = set(np.nonzero(m >= 0)[0])
    # transport to row r fails iff the fitted sin(phi) there exceeds 0.95; the fit equals the truth to ~1e-6
    must = {r for r in rows if s_of[r] < 0.949}
    never = {r for r in rows if s_of[r] > 0.951}
    assert must <= got and not (got & never) and len(never) >= 3


# ------------------------------------------------------------------------------------------- K4 (all 15), K6
def _kalman_update_matrix(p, C, i, m, e):
    """Textbook matrix-form update with H = e_i^T."""
    H = np.zeros((1, 5)); H[0, i] = 1.0
    S = float((H @ C @ H.T)[0, 0]) + e
    K = (C @ H.T) / S
    res = m - p[i]
    return p + K[:, 0] * res, C - K @ H @ C, res * res / S


@pytest.mark.parametrize("scale", [100.0, 7.0])
def test_turn_around_scales_all_15_and_whole_pass_structure(scale):
    """K1-K6 replayed on single smeared helices with the pinned transport (closed-form pins in test_oracle_units)
    and a matrix-form update: seed, chain + up pass through every row incl. the misses beyond the last hit, ONE
    transport back to lastRow, **C <- scale * C as a full matrix**, update with the lastRow hit, down pass through
    every row, misses below firstRow, ONE transport back to firstRow.  The oracle's output state must agree to
    1e-6 (fp64; scalar-form and matrix-form updates round differently on the inflated covariance, seen: 4e-8);
    scaling only the diagonal changes it at the 1e-3 level."""
    g = default_geometry()
    a = A_PER_KG * g.bz_kgauss
    rng = np.random.default_rng(31)
    b = single_track_events(6, rng, pt_range=(0.4, 3.0))
    prm = OracleParams(turn_cov_scale=scale)
    y64, z64 = b.y.astype(np.float64), b.z.astype(np.float64)
    res = oracle.track(g, y64, z64, b.row_offsets, b.n_tasks, precision="f64", params=prm, dump_tracklets=True)
    nr = g.n_rows
    X = g.row_x.astype(np.float64)
    tr = np.repeat(np.arange(len(b.row_offsets) - 1), np.diff(b.row_offsets.astype(np.int64)))
    n_checked = 0
    for t in range(res.n_tracks):
        hits = res.track_hits(t).astype(np.int64)
        rows = tr[hits] % nr
        k = np.nonzero(res.tracklet_nhits == len(hits))[0]
        k = [i for i in k if set(res.tracklet_map[i][res.tracklet_map[i] >= 0]) == set(hits)]
        if len(k) != 1 or len(hits) < 30:
            continue
        h0 = int(res.tracklet_start[k[0]])
        r0 = int(tr[h0] % nr)
        hit_of = dict(zip(rows.tolist(), hits.tolist()))
        assert r0 in hit_of and r0 + 1 in hit_of
        first, last = int(rows.min()), int(rows.max())
        # K1
        h1 = hit_of[r0 + 1]
        dx, dy, dz = X[r0 + 1] - X[r0], y64[h1] - y64[h0], z64[h1] - z64[h0]
        ri = 1.0 / np.sqrt(dx * dx + dy * dy)
        p = np.array([y64[h1], z64[h1], dy * ri, dz * ri, 0.0])
        C = np.diag([SY ** 2, SZ ** 2, 1.0, 1.0, 100.0])
        x = X[r0 + 1]

        def step(x, p, C, r):
            ok, x1, p1, c1 = oracle.transport(x, p, pack_cov(C), X[r], a)
            assert ok
            return x1, p1, unpack_cov(c1)

        def upd(p, C, h):
            p, C, c2a = _kalman_update_matrix(p, C, 0, y64[h], SY ** 2)
            p, C, c2b = _kalman_update_matrix(p, C, 1, z64[h], SZ ** 2)
            return p, C, c2a + c2b
        # K2 + K3: every row up to the row where the gap exceeds 4 (or the last row of the sector)
        gap, r = 0, r0 + 2
        while r < nr:
            x, p, C = step(x, p, C, r)
            if r in hit_of:
                p, C, _ = upd(p, C, hit_of[r]); gap = 0
            else:
                gap += 1
                if gap > 4:
                    break
            r += 1
        # K4
        if x != X[last]:
            x, p, C = step(x, p, C, last)
        C = C * scale
        p, C, chi2 = upd(p, C, hit_of[last])
        n_upd = 1
        # K5
        gap = 0
        for r in range(last - 1, -1, -1):
            x, p, C = step(x, p, C, r)
            if r in hit_of:
                p, C, c2 = upd(p, C, hit_of[r]); chi2 += c2; n_upd += 1
            elif r < first:
                gap += 1
                if gap > 4:
                    break
        # K6
        if x != X[first]:
            x, p, C = step(x, p, C, first)
        assert float(res.track_x[t]) == X[first]
        np.testing.assert_allclose(res.track_par[:, t], p, rtol=1e-6, atol=1e-9)
        np.testing.assert_allclose(unpack_cov(res.track_cov[:, t]), C, rtol=1e-5, atol=1e-12)
        np.testing.assert_allclose(res.track_chi2[t], chi2, rtol=1e-6)
        assert res.track_ndf[t] == 2 * n_upd - 5
        n_checked += 1
    assert n_checked >= 4


# ------------------------------------------------------------------------------------------- K7 / L1 tie
@pytest.mark.parametrize("b_first_in_start_row", [False, True])
def test_equal_length_tracklets_smaller_start_gid_owns_the_shared_cluster(b_first_in_start_row):
    """K7 (R16).  Two straight tracks A: y = +0.02 (x - x80) and B: y = -0.02 (x - x80) over rows 40..120 with ONE
    common cluster S = (0, z) in row 80.  S has two chi2 = 0 link pairs; the pair with the smaller up-gid wins
    (N5), here always A's (A is listed first in rows 79 and 81), so S is on A's CA chain and splits B's chain in two
    (start hits B41 and B81).  Three tracklets of 81 hits each contain S: A (start A41), B-lower (start B41, takes S
    by search at the predicted y = 0 exactly) and B-upper (start B81, takes S in its down pass).
    Equal nHits -> the SMALLER start gid owns: S goes to whichever of A41/B41 comes first in row 41, and B's own
    clusters to B-lower (B41 < B81).  Output: exactly two tracks, one with 81 hits holding S, one with 80."""
    g = G0
    x80 = float(g.row_x[80])
    pts = {}
    for r in range(40, 121):
        x = float(g.row_x[r])
        z = 0.5 * x
        if r == 80:
            pts[(0, r)] = [(0.0, z)]
            continue
        A, B = (0.02 * (x - x80), z), (-0.02 * (x - x80), z)
        pts[(0, r)] = [B, A] if (b_first_in_start_row and r == 41) else [A, B]
    gids = gid_table(pts)
    res = run(batch_from_rows(g, pts))
    S = gids[(80, 0)]
    a41 = gids[(41, 1 if b_first_in_start_row else 0)]
    b41 = gids[(41, 0 if b_first_in_start_row else 1)]
    b81 = gids[(81, 1)]
    # the premise: S is linked into A's chain, B's chain is split
    assert res.clean_up[S] == gids[(81, 0)] and res.clean_dn[S] == gids[(79, 0)]
    assert {a41, b41, b81} <= set(res.tracklet_start.tolist())
    for st in (a41, b41, b81):
        m = tracklet_from(res, st)
        assert (m >= 0).sum() == 81 and m[80] == S
    assert res.n_tracks == 2
    tracks = [set(res.track_hits(t).tolist()) for t in range(2)]
    with_s = [t for t in tracks if S in t]
    assert len(with_s) == 1 and len(with_s[0]) == 81
    other = [t for t in tracks if S not in t][0]
    assert len(other) == 80
    owner_start = b41 if b_first_in_start_row else a41
    assert owner_start in with_s[0], "equal length: the tracklet with the smaller start-hit gid owns S"
    assert (a41 if b_first_in_start_row else b41) in other


def test_longer_tracklet_owns_shared_clusters_whatever_the_gids():
    """K7: nHits decides before the gid.  B (rows 20..60, 41 hits) starts in a LOWER row than A (rows 40..158, 119
    hits), so every start hit of B has a smaller gid than A's (gids ascend with the row), and B is listed first in
    the common rows as well; they cross at row 50 in one common cluster - which the longer A must own."""
    g = G0
    x50 = float(g.row_x[50])
    pts = {}
    for r in range(20, 159):
        x = float(g.row_x[r])
        z = 0.5 * x
        A, B = (0.02 * (x - x50), z), (-0.02 * (x - x50), z)
        if r == 50:
            pts[(0, r)] = [(0.0, z)]
        elif r < 40:
            pts[(0, r)] = [B]
        elif r <= 60:
            pts[(0, r)] = [B, A]
        else:
            pts[(0, r)] = [A]
    gids = gid_table(pts)
    res = run(batch_from_rows(g, pts))
    S = gids[(50, 0)]
    b_lo = gids[(21, 0)]                                        # B's lower start hit
    assert tracklet_from(res, b_lo)[50] == S                    # B holds the common cluster ...
    a_trk = [i for i in range(res.n_tracklets) if res.tracklet_nhits[i] == 119]
    assert len(a_trk) >= 1                                      # (A's chain is split at S: two tracklets of A)
    for i in a_trk:
        assert res.tracklet_map[i][50] == S                     # ... and so does A
        assert int(res.tracklet_start[i]) > b_lo                # although A's start-hit gids are the larger ones
    lens = sorted(len(res.track_hits(t)) for t in range(res.n_tracks))
    assert lens == [40, 119]
    long_t = [t for t in range(res.n_tracks) if len(res.track_hits(t)) == 119][0]
    assert S in set(res.track_hits(long_t).tolist())
