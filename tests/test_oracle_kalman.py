"""Pins of the oracle's Kalman-filter steps (O4 Propagate / Update, SURVEY.md 8(c) "pins").

None of these re-types the oracle's formulas: Propagate is checked against the closed-form (asin)
helix and its finite-difference Jacobian, Update against the textbook matrix-form Kalman update done
with numpy.linalg, the fit against exact helix points and against numpy's polynomial least squares.
"""
import math

import numpy as np
import pytest

from oracle import tpc_oracle as orc
from tests.helpers import KAPPA, cov_to_full, full_to_cov, helix_step_closed_form, tri

BZ = 0.5


def _rand_states(n, seed, pt_min=0.08):
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        pt = math.exp(rng.uniform(math.log(pt_min), math.log(20.0)))
        q = rng.choice([-1.0, 1.0]) / pt
        s = rng.uniform(-0.85, 0.85)
        dx = rng.uniform(-3.2, 3.2)
        if abs(dx) < 0.05:
            continue
        if abs(s + dx * q * KAPPA * BZ) >= 0.95:
            continue
        out.append((np.array([rng.uniform(85, 245), rng.uniform(-40, 40), rng.uniform(-250, 250), s,
                              rng.uniform(-1.0, 1.0), q]), dx))
    return out


def test_propagate_matches_closed_form_helix_fp64():
    """fp64 instantiation vs the asin helix: <= 1e-9 relative (SURVEY.md 8(c) pins, row 'Propagate')."""
    worst = 0.0
    for st, dx in _rand_states(400, 11):
        ok, s1, _ = orc.propagate(st, np.zeros(15), st[0] + dx, BZ, 0.98, fp64=True)
        assert ok
        ref = helix_step_closed_form(st, dx, BZ)
        assert s1[0] == pytest.approx(ref[0], abs=1e-12)
        dy, dz = s1[1] - st[1], s1[2] - st[2]
        ry, rz = ref[1] - st[1], ref[2] - st[2]
        worst = max(worst, abs(dy - ry) / max(abs(ry), 1e-3), abs(dz - rz) / max(abs(rz), 1e-3),
                    abs(s1[3] - ref[3]))
        assert s1[4] == st[4] and s1[5] == st[5]
    assert worst < 1e-9


def test_propagate_straight_line_when_q_is_zero():
    """q = 0: y1 = y + dx*s/c, z1 = z + t*dx/c (closed form of a straight line)."""
    for s in (-0.7, -0.1, 0.0, 0.3, 0.9):
        for dx in (-2.0, 1.06, 3.0):
            st = np.array([100.0, 1.5, -20.0, s, 0.4, 0.0])
            ok, s1, _ = orc.propagate(st, np.zeros(15), 100.0 + dx, BZ, 0.98, fp64=True)
            assert ok
            c = math.sqrt(1 - s * s)
            assert s1[1] == pytest.approx(1.5 + dx * s / c, rel=1e-14, abs=1e-14)
            assert s1[2] == pytest.approx(-20.0 + 0.4 * dx / c, rel=1e-14)
            assert s1[3] == s


def test_propagate_conserves_circle_centre_and_radius():
    """In the bend plane the track is a circle: centre (x - s/k, y + c/k) and radius 1/|k| do not change."""
    st = np.array([85.0, 3.0, 10.0, 0.35, 0.7, -1.0 / 0.25])   # pT = 0.25 GeV/c
    k = st[5] * KAPPA * BZ
    cen0 = np.array([st[0] - st[3] / k, st[1] + math.sqrt(1 - st[3] ** 2) / k])
    cur = st.copy()
    for r in range(1, 60):
        ok, cur, _ = orc.propagate(cur, np.zeros(15), 85.0 + r * 1.06, BZ, 0.98, fp64=True)
        if not ok:
            break
        cen = np.array([cur[0] - cur[3] / k, cur[1] + math.sqrt(1 - cur[3] ** 2) / k])
        assert np.allclose(cen, cen0, rtol=0, atol=1e-9)
    assert r > 20


def test_propagate_fails_beyond_max_sinphi_and_leaves_state_alone():
    st = np.array([100.0, 0.0, 0.0, 0.97, 0.1, 1.0 / 0.05])
    cov = np.arange(15, dtype=float)
    ok, s1, c1 = orc.propagate(st, cov, 103.0, BZ, 0.98, fp64=True)
    assert not ok
    assert np.array_equal(s1, st) and np.array_equal(c1, cov)


def _jacobian_from_oracle(st, dx, fp64=True):
    """Column j of F = row j of F e_j e_j^T F^T (F_jj = 1); lower-triangle storage gives the upper part of F."""
    F = np.eye(5)
    for j in range(5):
        C = np.zeros((5, 5))
        C[j, j] = 1.0
        ok, _, c1 = orc.propagate(st, full_to_cov(C), st[0] + dx, BZ, 0.98, fp64=fp64)
        assert ok
        Cn = cov_to_full(c1)
        F[:, j] = Cn[j, :]
    return F


def _jacobian_fd(st, dx):
    """Central differences of the closed-form map; y = z = 0 (F does not depend on them) keeps the rounding noise low."""
    st = st.copy()
    st[1] = st[2] = 0.0
    F = np.zeros((5, 5))
    for j in range(5):
        h = 1e-4 * max(0.1, abs(st[1 + j]))
        a, b = st.copy(), st.copy()
        a[1 + j] += h
        b[1 + j] -= h
        d = helix_step_closed_form(a, dx, BZ, longdouble=True)[1:] - helix_step_closed_form(b, dx, BZ, longdouble=True)[1:]
        F[:, j] = (d / (2 * h)).astype(np.float64)
    return F


def test_propagate_jacobian_matches_finite_differences_of_the_closed_form():
    """Every element of F (incl. the Simpson form of F_zq) vs central differences of the asin helix.

    A dropped term, a wrong sign or a transposed index changes an element by O(its size); the analytic
    approximation error (series arc length, Simpson F_zq) stays below 1e-3 relative (measured worst 2.9e-4).
    """
    worst = 0.0
    for st, dx in _rand_states(200, 5):
        Fo = _jacobian_from_oracle(st, dx)
        Ff = _jacobian_fd(st, dx)
        # structure: identity + six upper elements
        mask = np.zeros((5, 5), bool)
        for (i, j) in ((0, 2), (0, 4), (1, 2), (1, 3), (1, 4), (2, 4)):
            mask[i, j] = True
        assert np.allclose(Fo[~mask], np.eye(5)[~mask], atol=1e-15)
        scale = np.maximum(np.abs(Ff), 1e-12)
        err = np.abs(Fo - Ff)[mask] / scale[mask]
        worst = max(worst, err.max())
    assert worst < 1e-3, worst


def test_propagate_covariance_is_F_C_Ft():
    """C' = F C F^T for a random symmetric positive C (numpy matmul as the reference)."""
    rng = np.random.default_rng(3)
    for st, dx in _rand_states(50, 9):
        A = rng.normal(size=(5, 5))
        C = A @ A.T + 0.1 * np.eye(5)
        F = _jacobian_from_oracle(st, dx)
        ok, _, c1 = orc.propagate(st, full_to_cov(C), st[0] + dx, BZ, 0.98, fp64=True)
        assert ok
        assert np.allclose(cov_to_full(c1), F @ C @ F.T, rtol=1e-11, atol=1e-12)


def test_update_equals_textbook_matrix_kalman_update():
    """Sequential scalar updates (y then z) == joint update with H = [I2 0], R = diag (numpy.linalg)."""
    rng = np.random.default_rng(17)
    H = np.zeros((2, 5))
    H[0, 0] = H[1, 1] = 1.0
    for _ in range(100):
        A = rng.normal(size=(5, 5))
        C = A @ A.T + 0.05 * np.eye(5)
        p = rng.normal(size=5)
        m = rng.normal(size=2)
        r = np.array([rng.uniform(0.005, 0.05), rng.uniform(0.005, 0.05)])
        st = np.concatenate([[100.0], p])
        ok, s1, c1, chi2 = orc.update(st, full_to_cov(C), 0.25, m[0], m[1], r[0], r[1], fp64=True)
        assert ok
        S = H @ C @ H.T + np.diag(r)
        K = C @ H.T @ np.linalg.inv(S)
        rho = m - H @ p
        p_ref = p + K @ rho
        C_ref = (np.eye(5) - K @ H) @ C
        chi_ref = 0.25 + rho @ np.linalg.solve(S, rho)
        assert np.allclose(s1[1:], p_ref, rtol=1e-10, atol=1e-12)
        assert np.allclose(cov_to_full(c1), C_ref, rtol=1e-9, atol=1e-12)
        assert chi2 == pytest.approx(chi_ref, rel=1e-10)
        assert s1[0] == 100.0


def test_update_rejects_non_positive_diagonal_and_non_finite():
    C = np.zeros(15)
    for i in range(5):
        C[tri(i, i)] = 1.0
    C[tri(4, 4)] = -1.0   # diagonal <= 0 after the update -> refused (R12)
    st = np.array([100.0, 0, 0, 0, 0, 0.0])
    ok, s1, c1, chi2 = orc.update(st, C, 0.0, 0.1, 0.1, 0.01, 0.01, fp64=True)
    assert not ok and np.array_equal(s1, st) and np.array_equal(c1, C) and chi2 == 0.0
    C[tri(4, 4)] = float("nan")
    ok, *_ = orc.update(st, C, 0.0, 0.1, 0.1, 0.01, 0.01, fp64=True)
    assert not ok


def _fit_points(xs, ys, zs, fp64, e2=0.01):
    """The constructor's fit sequence on given points: init from the first pair, filter up, turn, filter down."""
    dx, dy, dz = xs[1] - xs[0], ys[1] - ys[0], zs[1] - zs[0]
    L = math.sqrt(dx * dx + dy * dy)
    st = np.array([xs[0], ys[0], zs[0], dy / L, dz / L, 0.0])
    C = full_to_cov(np.diag([e2, e2, 1.0, 1.0, 100.0]))
    chi2 = 0.0
    for i in range(1, len(xs)):
        ok, st, C = orc.propagate(st, C, xs[i], BZ, 0.98, fp64)
        assert ok
        ok, st, C, chi2 = orc.update(st, C, chi2, ys[i], zs[i], e2, e2, fp64)
        assert ok
    C = full_to_cov(np.diag([100 * e2, 100 * e2, 1.0, 1.0, 100.0]))
    chi2 = 0.0
    for i in range(len(xs) - 1, -1, -1):
        ok, st, C = orc.propagate(st, C, xs[i], BZ, 0.98, fp64)
        assert ok
        ok, st, C, chi2 = orc.update(st, C, chi2, ys[i], zs[i], e2, e2, fp64)
        assert ok
    return st, C, chi2


def _exact_track(pt, s0, t, charge, y0=2.0, z0=-30.0, n=152):
    xs = 85.0 + np.arange(n) * (160.0 / 151.0)
    st = np.array([xs[0], y0, z0, s0, t, charge / pt])
    pts = [st]
    for i in range(1, n):
        nxt = helix_step_closed_form(pts[0], xs[i] - xs[0], BZ)
        if abs(nxt[3]) > 0.9:
            break
        pts.append(nxt)
    pts = np.array(pts)
    return xs[: len(pts)], pts


@pytest.mark.parametrize("pt,s0,t,charge", [(0.3, 0.2, 0.5, 1), (1.0, -0.3, -0.8, -1), (5.0, 0.1, 0.2, 1),
                                            (10.0, 0.0, 1.0, -1), (0.15, -0.1, 0.3, 1)])
def test_fit_of_exact_helix_points_recovers_the_parameters(pt, s0, t, charge):
    """BASELINE.json north_star check 3: exact helix points -> generating parameters to 1e-5 relative (fp64).

    fp32 is reported by SURVEY.md 8(c) as ~1-2e-5; asserted here at 2e-3 for q/pT (coordinate rounding
    alone is 4e-6 cm against a sagitta of a few mm at 10 GeV/c) and 1e-4 for the other parameters.
    """
    xs, pts = _exact_track(pt, s0, t, charge)
    assert len(xs) > 40
    st, C, chi2 = _fit_points(xs, pts[:, 1], pts[:, 2], fp64=True)
    truth = pts[0]
    floor = np.array([1.0, 1.0, 1.0, 1.0, abs(truth[5])])
    assert np.all(np.abs(st[1:] - truth[1:]) <= 1e-5 * np.maximum(np.abs(truth[1:]), floor)), (st, truth)
    assert chi2 < 1e-8
    st32, _, _ = _fit_points(xs, pts[:, 1], pts[:, 2], fp64=False)
    assert np.all(np.abs(st32[1:5] - truth[1:5]) <= 1e-4 * np.maximum(np.abs(truth[1:5]), 1.0))
    assert abs(st32[5] - truth[5]) <= 2e-3 * abs(truth[5]) + 2e-4


def test_fit_equals_weighted_least_squares_parabola_at_small_angles():
    """Special case with a textbook answer: at small angles y(x) is a parabola and z(x) a line, and with
    diffuse priors the filter is ordinary least squares -> compare with numpy.polyfit (library routine).
    """
    rng = np.random.default_rng(23)
    n = 60
    xs = 85.0 + np.arange(n) * (160.0 / 151.0)
    pt, charge = 8.0, 1.0
    k = charge / pt * KAPPA * BZ
    s0, t = 0.01, 0.05
    st0 = np.array([xs[0], 0.5, 3.0, s0, t, charge / pt])
    pts = np.array([helix_step_closed_form(st0, x - xs[0], BZ) for x in xs])
    ys = pts[:, 1] + rng.normal(0, 0.1, n)
    zs = pts[:, 2] + rng.normal(0, 0.1, n)
    st, C, chi2 = _fit_points(xs, ys, zs, fp64=True)
    u = xs - xs[0]
    cy = np.polyfit(u, ys, 2)     # y = y0 + s0*u + (k/2) u^2   (cos phi ~ 1)
    cz = np.polyfit(u, zs, 1)     # z = z0 + t*u
    # the prior (var 1 / 1 / 100 on s, t, q; 1 cm^2 on y, z) is ~1e4 x weaker than the data: agreement to a few 1e-4 of sigma
    sig = np.sqrt(np.array([C[tri(i, i)] for i in range(5)]))
    assert abs(st[1] - cy[2]) < 2e-2 * sig[0]
    assert abs(st[3] - cy[1]) < 2e-2 * sig[2]
    assert abs(st[5] * KAPPA * BZ - 2 * cy[0]) < 2e-2 * sig[4] * KAPPA * BZ
    assert abs(st[2] - cz[1]) < 2e-2 * sig[1]
    assert abs(st[4] - cz[0]) < 2e-2 * sig[3]
    # covariance of the straight-line z fit: textbook sigma^2 (X^T X)^-1
    X = np.stack([np.ones(n), u], 1)
    Vz = 0.01 * np.linalg.inv(X.T @ X)
    assert C[tri(1, 1)] == pytest.approx(Vz[0, 0], rel=2e-2)
    assert C[tri(3, 3)] == pytest.approx(Vz[1, 1], rel=2e-2)
    # chi2 of the down pass ~ residual sum of squares / sigma^2 of the two fits
    rss = np.sum((np.polyval(cy, u) - ys) ** 2 + (np.polyval(cz, u) - zs) ** 2) / 0.01
    assert chi2 == pytest.approx(rss, rel=5e-2)
