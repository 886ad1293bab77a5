"""Pins of the oracle's track model (docs/ARITH_SPEC.md section 5) - CPU only.

The transport is checked against the closed-form helix written with libm
(asin/cos), its Jacobian against finite differences of that closed form, the
covariance transport against a numpy matrix product, the scalar update against
the textbook matrix-form Kalman update.  None of these re-type the oracle's
sequence; each would fail on a dropped term, wrong sign or transposed index.
"""
import numpy as np
import pytest

import oracle
from helpers import A_PER_KG, helix_closed_form, pack_cov, unpack_cov

A = A_PER_KG * 5.0


def rand_state(rng, q_scale=3.0):
    p = np.array([rng.uniform(-20, 20), rng.uniform(5, 200), rng.uniform(-0.6, 0.6), rng.uniform(-1, 1),
                  rng.uniform(-q_scale, q_scale)])
    m = rng.standard_normal((5, 5))
    cov = m @ m.T * np.outer([0.1, 0.1, 0.01, 0.01, 0.5], [0.1, 0.1, 0.01, 0.01, 0.5])
    return p, cov


def test_transport_matches_closed_form_helix():
    rng = np.random.default_rng(1)
    for _ in range(300):
        p, cov = rand_state(rng, q_scale=10.0)  # down to pT = 0.1 GeV
        x = rng.uniform(85, 240)
        dx = rng.uniform(-4, 4)
        ok, x1, p1, _ = oracle.transport(x, p, pack_cov(cov), x + dx, A)
        ref = helix_closed_form(x, p, x + dx, A)
        if abs(ref[2]) > 0.95 or abs(p[2]) > 0.95:
            assert not ok
            continue
        assert ok and x1 == x + dx
        # arc length by 4-term asin series: relative error < 5e-7 (R13)
        np.testing.assert_allclose(p1, ref, rtol=1e-6, atol=1e-9)


def test_transport_straight_line_when_curvature_zero():
    p = np.array([1.0, 10.0, 0.3, 0.5, 0.0])
    ok, x1, p1, _ = oracle.transport(100.0, p, pack_cov(np.eye(5)), 103.0, A)
    c = np.sqrt(1 - 0.09)
    assert ok
    np.testing.assert_allclose(p1, [1.0 + 3.0 * 0.3 / c, 10.0 + 0.5 * 3.0 / c, 0.3, 0.5, 0.0], rtol=1e-14)


def test_transport_fails_beyond_max_sinphi_and_leaves_state():
    p = np.array([0.0, 0.0, 0.94, 0.0, -10.0])  # k = a*q > 0: sinphi grows with x
    c = pack_cov(np.eye(5))
    ok, x1, p1, c1 = oracle.transport(100.0, p, c, 102.0, A)
    assert not ok and x1 == 100.0
    np.testing.assert_array_equal(p1, p)
    np.testing.assert_array_equal(c1, c)


def test_transport_there_and_back_and_composition():
    rng = np.random.default_rng(2)
    for _ in range(100):
        p, cov = rand_state(rng)
        c = pack_cov(cov)
        x = 120.0
        ok, x1, p1, c1 = oracle.transport(x, p, c, x + 2.5, A)
        ok2, x2, p2, c2 = oracle.transport(x1, p1, c1, x, A)
        assert ok and ok2
        np.testing.assert_allclose(p2, p, rtol=1e-6, atol=1e-7)
        # covariance returns up to the first-order dz/dq entry (P19)
        np.testing.assert_allclose(unpack_cov(c2), cov, rtol=2e-2, atol=2e-3 * np.abs(cov).max())
        # x0 -> x1 -> x2 equals x0 -> x2 for the parameters
        oka, xa, pa, _ = oracle.transport(x1, p1, c1, x + 4.0, A)
        okb, xb, pb, _ = oracle.transport(x, p, c, x + 4.0, A)
        assert oka and okb
        np.testing.assert_allclose(pa, pb, rtol=1e-6, atol=1e-8)


def jacobian_from_oracle(x, p, xnew):
    """Column j of F = column j of C' when C = e_j e_j^T (F_jj = 1)."""
    F = np.zeros((5, 5))
    for j in range(5):
        cov = np.zeros((5, 5))
        cov[j, j] = 1.0
        ok, _, _, c1 = oracle.transport(x, p, pack_cov(cov), xnew, A)
        assert ok
        F[:, j] = unpack_cov(c1)[:, j]
    return F


def test_jacobian_matches_finite_differences_of_closed_form():
    rng = np.random.default_rng(3)
    for _ in range(50):
        p, _ = rand_state(rng, q_scale=5.0)
        x, xnew = 150.0, 150.0 + rng.choice([-1.0, 1.0]) * rng.uniform(0.5, 2.0)
        F = jacobian_from_oracle(x, p, xnew)
        Fd = np.zeros((5, 5))
        for j in range(5):
            # fd noise ~1e-16/(k*h): the q column (values ~1e-3, nearly linear in q) needs a wide step
            h = 1e-3 if j == 4 else 1e-5 * max(1.0, abs(p[j]))
            pp, pm = p.copy(), p.copy()
            pp[j] += h
            pm[j] -= h
            Fd[:, j] = (helix_closed_form(x, pp, xnew, A) - helix_closed_form(x, pm, xnew, A)) / (2 * h)
        exact = np.ones((5, 5), bool)
        exact[1, 4] = False  # dz/dq is first order in k*dx by design (P19)
        np.testing.assert_allclose(F[exact], Fd[exact], rtol=2e-6, atol=1e-9)
        assert abs(F[1, 4] - Fd[1, 4]) <= 0.15 * abs(Fd[1, 4]) + 1e-9
    # P19 converges to the exact derivative as dx -> 0
    p = np.array([1.0, 50.0, 0.4, 0.7, 2.0])
    errs = []
    for dx in (2.0, 0.5):
        F = jacobian_from_oracle(100.0, p, 100.0 + dx)
        h = 1e-6
        pp, pm = p.copy(), p.copy()
        pp[4] += h
        pm[4] -= h
        fd = (helix_closed_form(100.0, pp, 100.0 + dx, A)[1] - helix_closed_form(100.0, pm, 100.0 + dx, A)[1]) / (2 * h)
        errs.append(abs(F[1, 4] - fd) / abs(fd))
    assert errs[1] < errs[0]


def test_covariance_transport_is_F_C_Ft():
    rng = np.random.default_rng(4)
    for _ in range(50):
        p, cov = rand_state(rng)
        x, xnew = 100.0, 101.03
        F = jacobian_from_oracle(x, p, xnew)
        ok, _, _, c1 = oracle.transport(x, p, pack_cov(cov), xnew, A)
        np.testing.assert_allclose(unpack_cov(c1), F @ cov @ F.T, rtol=1e-10, atol=1e-14)


@pytest.mark.parametrize("i", [0, 1])
def test_update_is_textbook_kalman(i):
    rng = np.random.default_rng(5 + i)
    for _ in range(50):
        p, cov = rand_state(rng)
        m, e = p[i] + rng.normal(0, 0.3), 0.01 + rng.random() * 0.02
        p1, c1, chi2, ndf = oracle.update(p, pack_cov(cov), i, m, e, chi2=1.5, ndf=3)
        H = np.zeros((1, 5))
        H[0, i] = 1.0
        S = H @ cov @ H.T + e
        K = cov @ H.T / S
        np.testing.assert_allclose(p1, p + (K * (m - p[i])).ravel(), rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(unpack_cov(c1), (np.eye(5) - K @ H) @ cov, rtol=1e-10, atol=1e-14)
        assert ndf == 4
        np.testing.assert_allclose(chi2, 1.5 + (m - p[i]) ** 2 / S[0, 0], rtol=1e-12)


def test_f32_and_f64_instantiations_agree():
    rng = np.random.default_rng(7)
    for _ in range(50):
        p, cov = rand_state(rng)
        ok64, _, p64, c64 = oracle.transport(100.0, p, pack_cov(cov), 101.0, A)
        ok32, _, p32, c32 = oracle.transport(100.0, p.astype(np.float32), pack_cov(cov).astype(np.float32), 101.0,
                                             np.float32(A), precision="f32")
        assert ok64 == ok32
        np.testing.assert_allclose(p32, p64, rtol=2e-5, atol=2e-5)
        np.testing.assert_allclose(c32, c64, rtol=1e-3, atol=1e-5)
