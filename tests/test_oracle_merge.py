"""Pins of the oracle's O7 segment merger (NEXT-1 of SURVEY.md 8(f); DESIGN.md section 3 "O7", readings R31..R33).

Rotate is pinned against the closed-form helix seen from two sector frames (tests/helpers.truth_state_at_row, which
shares nothing with the oracle) and its covariance Jacobian against finite differences of that closed form; Match
against exact states on both sides of a sector border and of a row gap; the link rule against a brute-force
restatement in numpy; the whole pipeline against generator truth (every link joins segments of one generated
track) and against a constructed case where every track is cut in two by a band of removed rows.  CPU only.
"""
import math

import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen
from tests.helpers import cov_to_full, full_to_cov, helix_step_closed_form, truth_state_at_row

BZ = 0.5
A20 = math.radians(20.0)
ROW_X = (85.0 + np.arange(152) * (160.0 / 151.0)).astype(np.float32).astype(np.float64)


def _truth(pt, phi0, eta, h, sector, x):
    st = truth_state_at_row(pt, phi0, eta, 0.0, h, BZ, sector, x)
    return None if st is None else np.concatenate([[x], st])


@pytest.mark.parametrize("pt,h", [(0.4, 1), (0.4, -1), (2.0, 1), (8.0, -1)])
def test_rotate_equals_the_closed_form_helix_in_the_neighbour_frame(pt, h):
    """The same helix, seen from sector 3 and from sector 4: rotating the sector-3 state by +20 degrees gives a state at
    some plane x'; transporting the sector-4 truth to that plane (closed form) must give the same five parameters."""
    phi0 = math.radians(3.5 * 20.0 + 9.0)                      # close to the border between sectors 3 and 4
    for x in (100.0, 150.0, 200.0):
        a = _truth(pt, phi0, 0.4, h, 3, x)
        if a is None or abs(a[4]) > 0.7:
            continue
        ok, r, _ = orc.rotate(a, np.zeros(15), A20, fp64=True)
        assert ok
        b0 = _truth(pt, phi0, 0.4, h, 4, 120.0)
        assert b0 is not None
        b = helix_step_closed_form(b0, r[0] - b0[0], BZ)
        assert np.allclose(r[1:], b[1:], rtol=1e-9, atol=1e-9), (r, b)
        # and back
        ok, rr, _ = orc.rotate(r, np.zeros(15), -A20, fp64=True)
        assert ok and np.allclose(rr, a, rtol=1e-12, atol=1e-12)


def test_rotate_covariance_is_the_jacobian_of_the_closed_form():
    """C' = J C J^T with J = d(state at the turned plane) / d(state at the old plane), by central differences of
    'rotate the point and direction, then transport to the fixed new plane' in binary64."""
    rng = np.random.default_rng(3)

    def turned(st, alpha, xplane):       # exact: rotate position / direction, then closed-form transport to x' = xplane
        x, y, z, s, t, q = st
        ca, sa = math.cos(alpha), math.sin(alpha)
        c = math.sqrt(1 - s * s)
        r = np.array([x * ca + y * sa, y * ca - x * sa, z, s * ca - c * sa, t, q])
        return helix_step_closed_form(r, xplane - r[0], BZ)[1:]

    for alpha in (A20, -A20):
        for _ in range(20):
            st = np.array([rng.uniform(90, 240), rng.uniform(-20, 20), rng.uniform(-200, 200), rng.uniform(-0.5, 0.5),
                           rng.uniform(-1, 1), rng.uniform(-3, 3)])
            A = rng.normal(size=(5, 5))
            C = A @ A.T * 1e-3 + 1e-4 * np.eye(5)
            ok, r, c1 = orc.rotate(st, full_to_cov(C), alpha, fp64=True)
            assert ok
            J = np.zeros((5, 5))
            for j in range(5):
                d = np.zeros(6)
                hstep = 1e-6 * max(1.0, abs(st[1 + j]))
                d[1 + j] = hstep
                J[:, j] = (turned(st + d, alpha, r[0]) - turned(st - d, alpha, r[0])) / (2 * hstep)
            assert np.allclose(cov_to_full(c1), J @ C @ J.T, rtol=2e-5, atol=1e-9)


def test_rotate_refuses_beyond_max_sinphi():
    st = np.array([150.0, 0.0, 0.0, -0.9, 0.0, 0.0])           # sin(phi - 20 deg) < -0.98
    ok, r, c = orc.rotate(st, np.zeros(15), A20, fp64=True)
    assert not ok and np.array_equal(r, st)


def _diag_cov(sig):
    return full_to_cov(np.diag(np.asarray(sig, float) ** 2))


@pytest.mark.parametrize("rel", [0, 1, -1])
def test_match_of_exact_states_has_zero_chi2_and_displaced_states_the_textbook_chi2(rel):
    """Exact states of one helix at the two segment ends -> chi2 = 0; a known displacement d of b with diagonal
    covariances -> chi2 = sum d_i^2 / (sa_i^2 + sb_i^2) (closed form; the transported covariance is computed by the
    pinned Rotate / Propagate)."""
    pt, h, eta = 1.5, 1, 0.3
    sec_a = 5
    sec_b = sec_a + rel
    phi0 = math.radians((sec_a + 0.5) * 20.0 + 9.0 * rel)
    a = _truth(pt, phi0, eta, h, sec_a, ROW_X[60])
    b = _truth(pt, phi0, eta, h, sec_b, ROW_X[70])
    assert a is not None and b is not None
    tiny = _diag_cov([1e-3] * 5)
    ok, chi2 = orc.match(a, tiny, rel, b, tiny, BZ, fp64=True)
    assert ok and chi2 < 1e-9
    # transported covariance of a (by the oracle's own pinned steps), then a displaced b
    sa = _diag_cov([0.05, 0.08, 0.004, 0.006, 0.02])
    st, ca = a.copy(), sa.copy()
    if rel:
        ok, st, ca = orc.rotate(st, ca, A20 * rel, BZ, fp64=True)
    ok, st, ca = orc.propagate(st, ca, b[0], BZ, 0.98, True)
    sb = np.array([0.04, 0.07, 0.003, 0.005, 0.03])
    d = np.array([0.06, -0.1, 0.004, 0.0, -0.03])
    b2 = b.copy()
    b2[1:] += d
    ok, chi2 = orc.match(a, sa, rel, b2, _diag_cov(sb), BZ, fp64=True)
    var_a = np.array([ca[0], ca[2], ca[5], ca[9], ca[14]])
    assert ok and chi2 == pytest.approx(np.sum(d ** 2 / (var_a + sb ** 2)), rel=1e-6)
    # beyond the cut: refused
    b3 = b.copy()
    b3[1] += 5.0
    ok, _ = orc.match(a, sa, rel, b3, _diag_cov(sb), BZ, fp64=True)
    assert not ok


def _links_brute_force(res, n_sectors, p):
    """R31..R33 restated with numpy over all pairs, using only orc.match for the chi2 of a pair."""
    nt = res.n_tracks
    best_b, best_a = {}, {}
    for a in range(nt):
        if not res.rf_status[a]:
            continue
        for b in range(nt):
            if a == b or not res.rf_status[b]:
                continue
            sa, sb = int(res.trk_sector[a]), int(res.trk_sector[b])
            if sa == sb:
                rel = 0
            elif n_sectors == 36 and sa // 18 == sb // 18 and (sb % 18) == (sa % 18 + 1) % 18:
                rel = 1
            elif n_sectors == 36 and sa // 18 == sb // 18 and (sb % 18) == (sa % 18 + 17) % 18:
                rel = -1
            else:
                continue
            gap = int(res.trk_first_row[b]) - int(res.trk_last_row[a])
            if gap > p.merge_max_row_gap or gap < (1 if rel == 0 else -p.merge_back_rows):
                continue
            ok, chi2 = orc.match(np.concatenate([[res.rf_x_out[a]], res.rf_par_out[a]]), res.rf_cov_out[a], rel,
                                 np.concatenate([[res.rf_x_in[b]], res.rf_par_in[b]]), res.rf_cov_in[b], BZ, p, fp64=False)
            if not ok:
                continue
            if a not in best_b or (chi2, b) < best_b[a]:
                best_b[a] = (chi2, b)
            if b not in best_a or (chi2, a) < best_a[b]:
                best_a[b] = (chi2, a)
    nxt = np.full(nt, -1, np.int32)
    for a, (c, b) in best_b.items():
        if best_a[b][1] == a:
            nxt[a] = b
    return nxt


def test_links_equal_the_brute_force_restatement_and_are_reciprocal_chains():
    ev = datagen.make_event(1, scale=0.03)
    res = orc.run(ev, merge=True)
    assert res.n_tracks > 200 and (res.mg_next >= 0).sum() > 50
    nxt = _links_brute_force(res, ev.n_sectors, orc.default_params())
    assert np.array_equal(nxt, res.mg_next)
    has = res.mg_next >= 0
    idx = np.arange(res.n_tracks)
    assert np.array_equal(res.mg_prev[res.mg_next[has]], idx[has])          # reciprocity
    hp = res.mg_prev >= 0
    assert np.array_equal(res.mg_next[res.mg_prev[hp]], idx[hp])
    assert np.all(res.mg_head[~hp] == idx[~hp])                              # chain heads point to themselves
    assert np.array_equal(res.mg_head[has], res.mg_head[res.mg_next[has]])   # one head per chain
    assert np.all(res.mg_chi2[~has] == 0) and np.all(res.mg_chi2[has] <= 50.0)


def _majority_truth(ev, res, k):
    idx = res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]]
    t = ev.truth_track[idx]
    t = t[t >= 0]
    return -1 if len(t) == 0 else int(np.bincount(t).argmax())


def test_links_join_segments_of_the_same_generated_track():
    """Generator truth (not used by the oracle): on the Pb-Pb-like config, links across sector borders overwhelmingly
    join two segments of one generated particle, and most particles seen in two neighbouring sectors get linked."""
    ev = datagen.make_event(1, scale=0.05)
    res = orc.run(ev, merge=True)
    truth = np.array([_majority_truth(ev, res, k) for k in range(res.n_tracks)])
    a = np.nonzero(res.mg_next >= 0)[0]
    assert len(a) > 100
    same = truth[a] == truth[res.mg_next[a]]
    assert same.mean() > 0.97, same.mean()
    cross = res.trk_sector[a] != res.trk_sector[res.mg_next[a]]
    assert cross.sum() > 50                                                   # the sector-border case is exercised


def test_a_band_of_removed_rows_cuts_every_track_in_two_and_the_merger_rejoins_them():
    """Config 0 (one sector, 200 primaries) with the clusters of rows 70..79 removed: the constructor cannot bridge ten
    rows (max_row_gap = 4), so long tracks come out as two segments; the merger must link them (same truth track),
    and without the band there is nothing to link."""
    ev = datagen.make_event(0)
    whole = orc.run(ev, merge=True)
    assert (whole.mg_next >= 0).sum() <= 0.05 * whole.n_tracks
    off = ev.row_offset.astype(np.int64)
    keep = np.ones(ev.n_clusters, bool)
    keep[off[70]:off[80]] = False
    counts = np.diff(off)
    counts[70:80] = 0
    ev2 = datagen.event_from_arrays(np.concatenate([[0], np.cumsum(counts)]), ev.y[keep], ev.z[keep], 1, ev.n_rows)
    truth2 = ev.truth_track[keep]
    res = orc.run(ev2, merge=True)
    below = np.nonzero((res.trk_last_row < 70) & (res.trk_ncl >= 20))[0]
    above = np.nonzero((res.trk_first_row >= 80) & (res.trk_ncl >= 20))[0]
    assert len(below) > 50 and len(above) > 50

    def tr(k):
        idx = res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]]
        return int(np.bincount(truth2[idx][truth2[idx] >= 0]).argmax())
    t_above = {tr(k): k for k in above}
    n_pairs = n_linked = 0
    for k in below:
        partner = t_above.get(tr(k))
        if partner is None:
            continue
        n_pairs += 1
        n_linked += int(res.mg_next[k] == partner)
    assert n_pairs > 50 and n_linked >= 0.9 * n_pairs, (n_pairs, n_linked)
