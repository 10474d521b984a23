"""Pins of the oracle's O10 looper legs (rest of NEXT-1 of SURVEY.md 8(f); DESIGN.md section 3 "O10", readings
R40..R43; a looper is found as several legs, the two sides of a turn have to be joined).

Mirror is pinned by transport (the mirrored state walks the same helix backwards: closed form of tests/helpers, which
shares nothing with the oracle); LegMatch against exact states of both sides of a turn of a generated circle, in
sector frames up to four sectors apart; the pairing rule against a brute-force restatement in numpy on top of the
pinned single steps; the whole pipeline against generator truth.  CPU only.
"""
import itertools
import math

import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen
from tests.helpers import KAPPA, cov_to_full, helix_step_closed_form, sector_alpha, tri

BZ = 0.5
A20, A90 = math.radians(20.0), 0.5 * math.pi


def test_mirror_walks_the_same_helix_backwards():
    """M(state at x + dx) == transport of M(state at x) by -dx, for the closed-form helix."""
    rng = np.random.default_rng(11)
    for _ in range(50):
        st = np.array([rng.uniform(90, 240), rng.uniform(-30, 30), rng.uniform(-200, 200), rng.uniform(-0.8, 0.8),
                       rng.uniform(-1, 1), rng.uniform(-8, 8)])
        dx = rng.uniform(-10, 10)
        if abs(st[3] + dx * st[5] * KAPPA * BZ) > 0.95:
            continue
        st1 = helix_step_closed_form(st, dx, BZ)
        m0, _ = orc.mirror(st, np.zeros(15))
        m1, _ = orc.mirror(st1, np.zeros(15))
        assert m0[0] == -st[0] and m0[2] == st[2] and m0[3] == st[3]          # same z and inclination, opposite x
        assert np.allclose(helix_step_closed_form(m0, -dx, BZ), m1, rtol=1e-12, atol=1e-12)
        back, _ = orc.mirror(m0, np.zeros(15))
        assert np.array_equal(back, st)


def test_mirror_covariance_is_j_c_jt():
    rng = np.random.default_rng(12)
    A = rng.normal(size=(5, 5))
    C = A @ A.T
    c15 = np.array([C[i, j] for i in range(5) for j in range(i + 1)])
    st = np.array([150.0, 3.0, -20.0, 0.4, 0.7, -2.0])
    # J by differences of the (pinned) parameter map
    J = np.zeros((5, 5))
    for j in range(5):
        d = np.zeros(6); d[1 + j] = 1e-3
        J[:, j] = (orc.mirror(st + d, c15)[0][1:] - orc.mirror(st - d, c15)[0][1:]) / 2e-3
    assert np.allclose(J, np.diag([-1, 1, 1, -1, -1.0]), atol=1e-12)
    J = np.rint(J)
    _, m = orc.mirror(st, c15)
    assert np.array_equal(cov_to_full(m), J @ C @ J.T)


def _leg_state(pt, phi0, eta, vz, h, sector, x_row, back):
    """Forward-model state (x, y, z, s, t, q) of a generated circle at plane x_row of a sector frame: the outgoing crossing
    (back = False) or the returning one (back = True, direction reversed so that cos phi > 0: s, t and q change sign).
    Generator conventions as in tests/helpers.py: direction angle theta = delta - h*psi, sin(theta) = sin(delta) - h*x/R."""
    Rh = pt / (KAPPA * BZ)
    delta = phi0 - sector_alpha(sector)
    v = math.sin(delta) - h * x_row / Rh
    if abs(v) >= 1:
        return None
    theta = math.pi - math.asin(v) if back else math.asin(v)
    psi = h * (delta - theta)
    psi -= 2 * math.pi * math.floor(psi / (2 * math.pi))
    y = -h * Rh * (math.cos(delta) - math.cos(theta))
    tanl = math.sinh(eta)
    z = vz + Rh * psi * tanl
    q = -h / pt
    sign = -1.0 if back else 1.0
    return np.array([x_row, y, z, sign * v, sign * tanl, sign * q])


@pytest.mark.parametrize("h", [1, -1])
@pytest.mark.parametrize("d", [0, 1, 2, 3, 4])
def test_leg_match_of_the_two_sides_of_an_exact_turn(h, d):
    """A circle of pT = 100 MeV/c (R = 66.7 cm) that turns inside the TPC: its outgoing side seen from sector sa and its
    returning side seen from the sector d further on (in the direction the track moves) are matched with chi2 ~ 0;
    the same returning side one pitch later in z (the next turn of the helix), a flipped charge or a shifted position
    are refused or cost what the covariances say."""
    pt, eta, vz = 0.1, 0.3, 5.0
    sa = 5
    dsec = -h * d                                  # h = +1 turns towards smaller azimuth (theta = delta - psi)
    sb = (sa + dsec) % 18
    cov = np.zeros(15)
    for i in range(5):
        cov[tri(i, i)] = 1e-4
    found = centre_cut_seen = 0
    # off_deg: where the circle starts, relative to sector sa
    for off_deg, xa, xb in itertools.product(range(-90, 91, 15), (100.0, 110.0, 120.0, 125.0), (100.0, 112.0, 124.0)):
        phi0 = sector_alpha(sa) + math.radians(off_deg)
        a = _leg_state(pt, phi0, eta, vz, h, sa, xa, back=False)
        b = _leg_state(pt, phi0, eta, vz, h, sb, xb, back=True)
        if a is None or b is None or not (0.5 <= abs(a[3]) < 0.97 and 0.5 <= abs(b[3]) < 0.97) or a[3] * b[3] >= 0:
            continue
        if (a[3] > 0) != (dsec >= 0) and dsec != 0:
            continue
        ok, chi2 = orc.leg_match(a, cov, dsec, b, cov, BZ, fp64=True)
        if not ok:
            continue                            # a turned frame too steep for Propagate: allowed to refuse
        found += 1
        assert chi2 < 1e-6, (xa, xb, chi2)         # arc-length series over eight steps: ~1e-7 cm in z
        # the pair is symmetric in its roles: b as the propagated one, a the other, sector distance reversed
        ok2, chi2b = orc.leg_match(b, cov, -dsec, a, cov, BZ, fp64=True)
        assert ok2 and chi2b < 1e-6
        # next turn of the helix: same circle, z one pitch further -> only the z term, far above the cut
        b2 = b.copy(); b2[2] += 2 * math.pi * (pt / (KAPPA * BZ)) * math.sinh(eta)
        assert not orc.leg_match(a, cov, dsec, b2, cov, BZ, fp64=True)[0]
        p = orc.default_params(); p.leg_chi2_max = 1e30
        ok3, c3 = orc.leg_match(a, cov, dsec, b2, cov, BZ, p, fp64=True)
        assert ok3 and c3 > 1e3
        # a mismatch of dz in z alone costs dz^2 / (C11_a' + C11_b) with C11_a' >= C11_a (transport only adds variance)
        b3 = b.copy(); b3[2] += 0.05
        ok4, c4 = orc.leg_match(a, cov, dsec, b3, cov, BZ, p, fp64=True)
        assert ok4 and 1e-6 < c4 <= 0.05 ** 2 / 2e-4 * (1 + 1e-9)
        cz = np.zeros(15); cz[tri(1, 1)] = 1e-4                      # z variance only: nothing is added to it
        ok5, c5 = orc.leg_match(a, cz, dsec, b3, cz, BZ, p, fp64=True)
        assert not ok5                                                # zero denominators of the other terms refuse (R32)
        cy = cov.copy(); cy[tri(3, 3)] = 0.0                          # no dip variance: C11_a' = C11_a + jz^2 C00 >= 1e-4
        ok6, c6 = orc.leg_match(a, cy, dsec, b3, cov, BZ, p, fp64=True)
        assert ok6 and c6 >= c4
        # R44: the circle centres of the two sides must be close: b moved sideways by 3 cm moves its centre by 3 cm
        b4 = b.copy(); b4[1] += 3.0
        verdict = {}
        for cut in (2.9, 3.1, 1e9):
            p4 = orc.default_params(); p4.leg_chi2_max = 1e30; p4.leg_max_centre_dist = cut
            verdict[cut] = orc.leg_match(a, cov, dsec, b4, cov, BZ, p4, fp64=True)[0]
        assert not verdict[2.9] and verdict[3.1] == verdict[1e9]
        centre_cut_seen += verdict[3.1]
        # wrong charge or wrong dip on one side (what a missing sign in Mirror would look like)
        for idx in (4, 5):
            bw = b.copy(); bw[idx] = -bw[idx]
            okw, cw = orc.leg_match(a, cov, dsec, bw, cov, BZ, p, fp64=True)
            assert (not okw) or cw > 100.0
    assert found >= 2 and centre_cut_seen >= 1


def _legs_numpy(ev, res, p):
    """O10 restated on top of the pinned single steps (orc.rotate, orc.propagate in binary32; Mirror by numpy signs)."""
    nt = res.n_tracks
    msp = p.max_sinphi
    f32 = np.float32

    def outer(k):
        return np.concatenate([[res.rf_x_out[k]], res.rf_par_out[k]]), res.rf_cov_out[k].copy()

    def centre(st):                                  # circle centre of a state in its own frame, binary32 step by step
        x, y, s, q = f32(st[0]), f32(st[1]), f32(st[3]), f32(st[5])
        k = q * f32(KAPPA * ev.bz_tesla)
        return x - s / k, y + np.sqrt(f32(1) - s * s) / k

    def chi2_of(a, b, d):
        (A, CA), (B, CB) = outer(a), outer(b)
        with np.errstate(all="ignore"):
            (xa, ya), (xb, yb) = centre(A), centre(B)
            cd, sd = f32(math.cos(d * 2.0 * 0.17453292519943295)), f32(math.sin(d * 2.0 * 0.17453292519943295))
            ex, ey = (xb * cd - yb * sd) - xa, (xb * sd + yb * cd) - ya
            md = f32(p.leg_max_centre_dist)
            if not ex * ex + ey * ey <= md * md:
                return None
        sg = 1.0 if A[3] > 0 else -1.0
        alpha = d * math.radians(10.0) + sg * A90
        oka, A, CA = orc.rotate(A, CA, alpha, ev.bz_tesla, msp, fp64=False)
        okb, B, CB = orc.rotate(B, CB, -alpha, ev.bz_tesla, msp, fp64=False)
        if not (oka and okb):
            return None
        B[0], B[1], B[4], B[5] = -B[0], -B[1], -B[4], -B[5]            # Mirror (the diagonal of C is unchanged)
        x0, step = f32(A[0]), (f32(B[0]) - f32(A[0])) * f32(0.125)
        for i in range(1, 9):
            ok, A, CA = orc.propagate(A, CA, float(x0 + f32(i) * step) if i < 8 else B[0], ev.bz_tesla, msp, fp64=False)
            if not ok:
                return None
        tot = f32(0)
        for i in range(5):
            den = f32(CA[tri(i, i)]) + f32(CB[tri(i, i)])
            if not den > 0:
                return None
            dd = f32(A[1 + i]) - f32(B[1 + i])
            tot = tot + (dd * dd) / den
        return tot if tot <= f32(p.leg_chi2_max) else None

    ends = [k for k in range(nt) if res.rf_status[k] and not (abs(f32(res.rf_par_out[k, 2])) < f32(p.leg_min_sinphi))]
    best = {}
    for ia, a in enumerate(ends):
        for b in ends[ia + 1:]:
            sa, sb = int(res.trk_sector[a]), int(res.trk_sector[b])
            if sa == sb:
                d = 0
            elif ev.n_sectors == 36 and sa // 18 == sb // 18:
                d = (sb % 18 - sa % 18) % 18
                d = d - 18 if d > 9 else d
            else:
                continue
            if abs(d) > p.leg_max_sectors or abs(int(res.trk_last_row[a]) - int(res.trk_last_row[b])) > p.leg_max_row_diff:
                continue
            s_a, s_b = res.rf_par_out[a, 2], res.rf_par_out[b, 2]
            if not s_a * s_b < 0 or (s_a > 0 and d < 0) or (s_a < 0 and d > 0):
                continue
            c = chi2_of(a, b, d)
            if c is None:
                continue
            for u, v in ((a, b), (b, a)):
                if u not in best or (c, v) < best[u]:
                    best[u] = (c, v)
    partner, chi2 = np.full(nt, -1, np.int32), np.zeros(nt)
    for k, (c, o) in best.items():
        if best.get(o, (0, -1))[1] == k:
            partner[k], chi2[k] = o, float(c)
    return partner, chi2


@pytest.mark.parametrize("scale,dead,centre,least", [(0.05, (), 10.0, 20), (0.04, (30, 31, 90), 10.0, 20), (0.05, (), 0.7, 4)])
def test_legs_equal_the_numpy_restatement(scale, dead, centre, least):
    ev = datagen.make_event(2, scale=scale, dead_rows=dead)
    p = orc.default_params()
    p.leg_max_centre_dist = centre
    res = orc.run(ev, p, legs=True)
    partner, chi2 = _legs_numpy(ev, res, p)
    assert (partner >= 0).sum() >= least
    if centre < 1.0:                                 # the tight cut really bites: fewer pairs than with the default
        assert (partner >= 0).sum() < 0.8 * (orc.run(ev, legs=True).lg_partner >= 0).sum()
    assert np.array_equal(partner, res.lg_partner)
    assert np.array_equal(chi2, res.lg_chi2)


def test_legs_join_the_two_sides_of_generated_turns():
    """Generator truth (config 2: loopers of 50-150 MeV/c): every pair joins two tracks of one generated particle and of
    one turn of its helix; the rule's own invariants; and most turns that left two steep ends are found."""
    ev = datagen.make_event(2, scale=0.1)
    p = orc.default_params()
    res = orc.run(ev, p, legs=True)
    nt = res.n_tracks
    lp = res.lg_partner

    def majority(arr, k):
        v = arr[res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]]]
        return np.bincount(v + 1).argmax() - 1

    truth = np.array([majority(ev.truth_track, k) for k in range(nt)])
    turn = np.array([majority(ev.truth_turn, k) for k in range(nt)])
    linked = np.nonzero(lp >= 0)[0]
    assert len(linked) >= 300 and len(linked) % 2 == 0
    assert np.array_equal(lp[lp[linked]], linked)                                  # pairs
    assert np.all(truth[linked] == truth[lp[linked]]) and np.all(truth[linked] >= 0)
    assert np.all(turn[linked] == turn[lp[linked]])                                # not the next turn of the helix
    s_out = res.rf_par_out[:, 2]
    assert np.all(s_out[linked] * s_out[lp[linked]] < 0) and np.all(np.abs(s_out[linked]) >= 0.5)
    assert np.all(np.abs(res.trk_last_row[linked] - res.trk_last_row[lp[linked]]) <= p.leg_max_row_diff)
    assert np.all(res.trk_sector[linked] // 18 == res.trk_sector[lp[linked]] // 18)
    assert np.all(res.lg_chi2[linked] <= p.leg_chi2_max) and np.all(res.lg_chi2[lp < 0] == 0)
    assert np.array_equal(res.lg_chi2[linked], res.lg_chi2[lp[linked]])
    # efficiency: (particle, turn) groups with a steep end of each inclination, whose outermost ends are within the
    # row window -> at least 80 % of them carry a link
    ends = (res.rf_status == 1) & (np.abs(s_out) >= 0.5) & (truth >= 0)
    groups = {}
    for k in np.nonzero(ends)[0]:
        groups.setdefault((truth[k], turn[k]), []).append(k)
    want = got = 0
    for ks in groups.values():
        pos = [k for k in ks if s_out[k] > 0]
        neg = [k for k in ks if s_out[k] < 0]
        if not pos or not neg:
            continue
        a = max(pos, key=lambda k: res.trk_last_row[k]); b = max(neg, key=lambda k: res.trk_last_row[k])
        if abs(int(res.trk_last_row[a]) - int(res.trk_last_row[b])) > p.leg_max_row_diff:
            continue
        want += 1
        got += any(lp[k] >= 0 for k in ks)
    assert want >= 100 and got >= 0.8 * want, (want, got)


def test_legs_leave_the_other_outputs_alone_and_straight_tracks_unpaired():
    ev = datagen.make_event(1, scale=0.03)
    plain = orc.run(ev, refit=True)
    res = orc.run(ev, legs=True)
    assert np.array_equal(plain.trk_cl_index, res.trk_cl_index) and np.array_equal(plain.rf_par_out, res.rf_par_out)
    hi_pt = np.abs(res.rf_par_out[:, 4]) < 1.0                     # pT > 1 GeV/c: R > 6.7 m, no turn inside the TPC
    assert hi_pt.sum() > 50 and np.all(res.lg_partner[hi_pt] == -1)
