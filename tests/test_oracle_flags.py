"""Pins of the oracle's O8 cluster flags (NEXT-3 of SURVEY.md 8(f); DESIGN.md section 3 "O8"; PAPER.md L77-L90:
adjacent = within a tube of 1.5 cm, ambiguity to the higher-momentum track; protected = adjacent to a track with
pT > 50 MeV/c and |phi| < 70 deg; strategy B removes everything unprotected, strategy A the unprotected clusters
attached or adjacent to a low-pT / steep track).

Hand-built cases with known distances and momenta, a numpy restatement of the rule on top of the pinned single
Propagate step, the truth table of the flag bits, and set invariants.  CPU only.
"""
import math

import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen
from tests.helpers import helix_step_closed_form

BZ = 0.5
R = 152
ROW_X = (85.0 + np.arange(R) * (160.0 / 151.0)).astype(np.float32).astype(np.float64)
ATT, ADJ, PROT, RMA, RMB = 1, 2, 4, 8, 16


def _event(points):
    """points: list of (row, y, z) -> one-sector Event; returns (event, index of every point in the CSR order)."""
    pts = sorted(enumerate(points), key=lambda t: t[1][0])
    rows = np.array([p[1][0] for p in pts])
    counts = np.bincount(rows, minlength=R)
    off = np.concatenate([[0], np.cumsum(counts)])
    ev = datagen.event_from_arrays(off, np.array([p[1][1] for p in pts], np.float32), np.array([p[1][2] for p in pts], np.float32), 1, R)
    where = np.empty(len(points), int)
    for pos, (orig, _) in enumerate(pts):
        where[orig] = pos
    return ev, where


def _helix_points(pt, charge, s0, t, y0, z0, rows):
    st0 = np.array([ROW_X[rows[0]], y0, z0, s0, t, charge / pt])
    return [helix_step_closed_form(st0, ROW_X[r] - ROW_X[rows[0]], BZ) for r in rows]


def test_tube_radius_on_a_hand_built_track():
    """Exact straight-ish track (pT = 20 GeV/c) plus four extra clusters on row 30 at known distances from it."""
    rows = list(range(10, 70))
    tr = _helix_points(20.0, 1, 0.1, 0.3, -3.0, 20.0, rows)
    pts = [(r, p[1], p[2]) for r, p in zip(rows, tr)]
    y30, z30 = tr[20][1], tr[20][2]
    extra = [(30, y30 + 1.4, z30), (30, y30 - 1.6, z30), (30, y30 + 1.0, z30 - 1.0), (30, y30 - 1.1, z30 + 1.1)]
    ev, where = _event(pts + extra)
    res = orc.run(ev, flags=True)
    assert res.n_tracks == 1 and res.trk_ncl[0] == len(rows)
    f = res.cf_flags
    assert np.all(f[where[:len(rows)]] == ATT | ADJ | PROT)
    e = where[len(rows):]
    assert f[e[0]] == ADJ | PROT and f[e[2]] == ADJ | PROT           # 1.4 cm and sqrt(2) cm: inside the tube
    assert f[e[1]] == RMB and f[e[3]] == RMB                          # 1.6 cm and 1.1 * sqrt(2) cm: outside
    assert np.all(res.cf_owner[where[:len(rows)]] == 0) and res.cf_owner[e[0]] == 0 and res.cf_owner[e[1]] == -1
    # track-model residuals (R39): exact helix points leave none (fp32 rounding only), unattached clusters carry 0
    assert np.all(np.abs(res.cf_res_y[where[:len(rows)]]) < 2e-4) and np.all(np.abs(res.cf_res_z[where[:len(rows)]]) < 2e-4)
    assert np.all(res.cf_res_y[e] == 0) and np.all(res.cf_res_z[e] == 0)


def test_ambiguity_goes_to_the_higher_momentum_track_and_low_momentum_tracks_do_not_protect():
    rows = list(range(5, 45))         # short enough that the different curvatures keep the two tracks > 1.5 cm apart
    a = _helix_points(2.0, 1, 0.0, 0.2, 0.0, 10.0, rows)            # 2 GeV/c
    b = _helix_points(6.0, 1, 0.0, 0.2, 2.5, 10.0, rows)            # 6 GeV/c, 2.5 cm beside it
    pts = [(r, p[1], p[2]) for r, p in zip(rows, a)] + [(r, p[1], p[2]) for r, p in zip(rows, b)]
    mid = [(r, 0.5 * (a[i][1] + b[i][1]), a[i][2]) for i, r in enumerate(rows) if 8 <= r <= 12]      # in both tubes
    ev, where = _event(pts + mid)
    res = orc.run(ev, flags=True)
    assert res.n_tracks == 2
    pt = 1.0 / np.abs(res.rf_par_in[:, 4])
    hi = int(np.argmax(pt))
    assert pt[hi] == pytest.approx(6.0, rel=0.05) and pt[1 - hi] == pytest.approx(2.0, rel=0.05)
    m = where[2 * len(rows):]
    assert np.all(res.cf_owner[m] == hi) and np.all(res.cf_flags[m] == ADJ | PROT)
    # the tracks own their clusters (2.5 cm apart: outside each other's tube)
    assert np.all(res.cf_owner[where[:len(rows)]] == 1 - hi) and np.all(res.cf_owner[where[len(rows):2 * len(rows)]] == hi)
    # protect only above 4 GeV/c: the 2 GeV/c track now marks its clusters for removal by strategy A
    p = orc.default_params()
    p.inv_pt_protect = 0.25
    res = orc.run(ev, p, flags=True)
    assert np.all(res.cf_flags[where[:len(rows)]] == ATT | ADJ | RMA | RMB)
    assert np.all(res.cf_flags[where[len(rows):2 * len(rows)]] == ATT | ADJ | PROT)
    assert np.all(res.cf_flags[m] == ADJ | PROT)                     # still owned by the 6 GeV/c track


def _flags_numpy(ev, res, p, rank=None):
    """O8 restated: walk every refitted track with the pinned single Propagate step (binary32), tubes by numpy.
    rank: leg rank per track (1 = secondary leg: it does not protect), None = every track is a primary leg."""
    n = ev.n_clusters
    off = ev.row_offset.astype(np.int64)
    rowof = np.repeat(np.arange(ev.n_rows * ev.n_sectors), np.diff(off)) % ev.n_rows
    owner = np.full(n, -1, np.int64)
    oq = np.zeros(n, np.float32)
    good_any = np.zeros(n, bool)                 # R36b: some good track has the cluster in its tube
    res_y, res_z = np.zeros(n), np.zeros(n)
    sin70 = np.float32(0.9396926207859084)
    tube2 = np.float32(p.tube_radius) * np.float32(p.tube_radius)
    y32, z32 = ev.y.astype(np.float32), ev.z.astype(np.float32)
    row_x = np.asarray(ev.row_x, np.float32).astype(np.float64)
    for k in range(res.n_tracks):
        if not res.rf_status[k]:
            continue
        st = np.concatenate([[res.rf_x_in[k]], res.rf_par_in[k]])
        cov = res.rf_cov_in[k].copy()
        aq = np.float32(abs(st[5]))
        low = not (aq < np.float32(p.inv_pt_protect))
        cl = res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]].astype(np.int64)
        sec = int(res.trk_sector[k])
        for r in range(int(res.trk_first_row[k]), int(res.trk_last_row[k]) + 1):
            if ev.row_dead[r]:
                continue
            if r > res.trk_first_row[k]:
                ok, st, cov = orc.propagate(st, cov, row_x[r], ev.bz_tesla, p.max_sinphi, fp64=False)
                if not ok:
                    break
            lo, hi = off[sec * ev.n_rows + r], off[sec * ev.n_rows + r + 1]
            dy = y32[lo:hi] - np.float32(st[1])
            dz = z32[lo:hi] - np.float32(st[2])
            inside = (dy * dy + dz * dz) <= tube2
            if p.tube_chi2_max > 0:                      # R49
                c32 = cov.astype(np.float32)
                x2 = (dy * dy) / (c32[0] + np.float32(p.err2_y)) + (dz * dz) / (c32[2] + np.float32(p.err2_z))
                inside &= x2 <= np.float32(p.tube_chi2_max)
            own = cl[rowof[cl] == r]
            inside[own - lo] = True
            for c in own:
                res_y[c] = float(y32[c] - np.float32(st[1]))
                res_z[c] = float(z32[c] - np.float32(st[2]))
            b = low or not (np.float32(abs(st[3])) < sin70) or (rank is not None and rank[k] == 1)
            for c in np.nonzero(inside)[0] + lo:
                good_any[c] |= not b
                if owner[c] < 0 or aq < oq[c]:
                    owner[c], oq[c] = k, aq
    f = np.zeros(n, np.uint8)
    f[res.trk_cl_index] |= ATT
    has = owner >= 0
    prot = has & good_any
    f[has] |= ADJ
    f[prot] |= PROT
    f[has & ~prot] |= RMA
    f[~prot] |= RMB
    return f, owner, res_y, res_z


@pytest.mark.parametrize("idx,scale,dead", [(2, 0.03, ()), (1, 0.02, (40, 97))])
def test_flags_equal_the_numpy_restatement(idx, scale, dead):
    ev = datagen.make_event(idx, scale=scale, dead_rows=dead)
    p = orc.default_params()
    res = orc.run(ev, p, flags=True)
    f, owner, ry, rz = _flags_numpy(ev, res, p)
    assert np.array_equal(owner, res.cf_owner)
    assert np.array_equal(f, res.cf_flags)
    assert np.array_equal(ry, res.cf_res_y) and np.array_equal(rz, res.cf_res_z)
    if idx == 2:
        assert ((res.cf_flags & RMA) != 0).sum() > 10            # steep looper segments are exercised
        # with the leg labels of O12: secondary legs do not protect and are removable by strategy A (L86)
        res = orc.run(ev, p, flags=True, merged=True)
        assert (res.mt_rank == 1).sum() > 5
        f2, owner2, _, _ = _flags_numpy(ev, res, p, rank=res.mt_rank)
        assert np.array_equal(owner2, res.cf_owner) and np.array_equal(owner2, owner)      # ownership does not look at legs
        assert np.array_equal(f2, res.cf_flags)
        assert ((f2 & RMA) != 0).sum() > ((f & RMA) != 0).sum() + 100


def test_every_good_track_protects_the_clusters_in_its_tube_even_when_a_steep_track_owns_them():
    """R36b ("All clusters adjacent to the primary leg of a track with pT > 50 MeV/c and |phi| < 70 degrees
    are protected"; L88: strategy A "only rejects clusters that have been positively identified as not useful").  Two exact
    circles in one sector: G with pT = 70 MeV/c at moderate angles, and S with pT = 120 MeV/c whose sin(phi) passes
    sin(70 degrees) = 0.94 between rows 43 and 44 (0.5 + 0.012491 / cm * 1.0596 cm * (row - 10): 0.937, 0.950).  G is laid 0.5 cm
    beside S on row 45.  By hand: S has the higher momentum, so it owns the clusters of both tracks that lie in its tube on row 45; it is steep there, so it protects nothing -- but G is a good
    track and those clusters are in G's own tube: they stay protected (flags attached | adjacent | protected, owner = S).
    Under the round-1 reading (protection only through the owner) they were removed by strategies A and B."""
    b_field = 0.00299792458 * BZ

    def circle(pt, s10, y10, z10, t, rows, y_at=None):
        k = (1.0 / pt) * b_field
        s_of = lambda r: s10 + k * (ROW_X[r] - ROW_X[10])
        c10 = math.sqrt(1 - s10 * s10)
        ys = {r: y10 + (c10 - math.sqrt(1 - s_of(r) ** 2)) / k for r in rows}
        zs = {r: z10 + t * (math.asin(s_of(r)) - math.asin(s10)) / k for r in rows}
        return s_of, ys, zs

    rows_s = list(range(10, 47))
    sS, yS, zS = circle(0.12, 0.50, 0.0, 30.0, 0.3, rows_s)
    assert sS(43) < 0.9397 < sS(44) and sS(46) < 0.98                       # steep from row 44 on, inside max_sinphi
    rows_g = list(range(10, 60))
    sG, yG0, zG0 = circle(0.07, -0.45, 0.0, 0.0, 0.25, rows_g)
    dy, dz = yS[45] + 0.4 - yG0[45], zS[45] + 0.3 - zG0[45]                 # shift G so that it passes 0.5 cm from S on row 45
    pts = [(r, yS[r], zS[r]) for r in rows_s] + [(r, yG0[r] + dy, zG0[r] + dz) for r in rows_g]
    ev, where = _event(pts)
    res = orc.run(ev, flags=True)
    assert res.n_tracks == 2
    pt = 1.0 / np.abs(res.rf_par_in[:, 4])
    kS, kG = int(np.argmax(pt)), int(np.argmin(pt))
    assert pt[kS] == pytest.approx(0.12, rel=0.05) and pt[kG] == pytest.approx(0.07, rel=0.05)
    g45 = where[len(rows_s) + (45 - 10)]
    s45 = where[45 - 10]
    assert res.cf_owner[g45] == kS and res.cf_owner[s45] == kS             # the higher-momentum track owns both
    assert res.cf_flags[g45] == ATT | ADJ | PROT                           # ... but G protects what is in its tube
    assert res.cf_flags[s45] == ATT | ADJ | PROT                           # S's own cluster lies 0.5 cm from G as well
    far = where[46 - 10]                                                   # S on row 46: steep, and G is > 1.5 cm away by then
    g_at_46 = np.hypot(yS[46] - (yG0[46] + dy), zS[46] - (zG0[46] + dz))
    assert g_at_46 > 1.6
    assert res.cf_flags[far] == ATT | ADJ | RMA | RMB and res.cf_owner[far] == kS


def test_flag_invariants_and_what_the_strategies_remove():
    ev = datagen.make_event(2, scale=0.05)
    res = orc.run(ev, flags=True)
    f = res.cf_flags
    att, adj, prot, rma, rmb = ((f & b) != 0 for b in (ATT, ADJ, PROT, RMA, RMB))
    assert np.array_equal(adj, res.cf_owner >= 0)
    assert not np.any(prot & ~adj) and not np.any(rma & ~adj)
    assert np.array_equal(rmb, ~prot) and np.array_equal(rma, adj & ~prot)
    refitted = res.rf_status[np.repeat(np.arange(res.n_tracks), res.trk_ncl)] == 1
    assert np.all(adj[res.trk_cl_index[refitted]])                  # attached clusters of refitted tracks count as adjacent
    # strategy A never removes a cluster no track claims; strategy B removes all of those (noise included)
    noise = ev.truth_track < 0
    assert rmb[noise & ~adj].all() and not rma[~adj].any()
    # most noise is far from any track and most track clusters are protected
    assert prot[~noise].mean() > 0.7 and rmb[noise].mean() > 0.6


def test_residuals_have_the_least_squares_variance():
    """Closed form: residuals of a least-squares fit with p free parameters over n points of variance sigma^2 have the
    variance sigma^2 (1 - p / n); the helix has 3 parameters in the bend plane (y) and 2 in z.  Config 0: sigma = 0.1 cm."""
    ev = datagen.make_event(0)
    res = orc.run(ev, flags=True)
    long_tracks = np.nonzero((res.rf_status == 1) & (res.trk_ncl >= 40))[0]
    ry, rz, ey, ez = [], [], [], []
    for k in long_tracks:
        idx = res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]]
        n = len(idx)
        ry.append(res.cf_res_y[idx]); rz.append(res.cf_res_z[idx])
        ey.append(np.full(n, 0.01 * (1 - 3.0 / n))); ez.append(np.full(n, 0.01 * (1 - 2.0 / n)))
    ry, rz, ey, ez = (np.concatenate(a) for a in (ry, rz, ey, ez))
    assert len(ry) > 8000
    assert np.mean(ry ** 2) == pytest.approx(np.mean(ey), rel=0.05)
    assert np.mean(rz ** 2) == pytest.approx(np.mean(ez), rel=0.05)
    assert abs(np.mean(ry)) < 0.005 and abs(np.mean(rz)) < 0.005


def test_chi2_tube_on_a_hand_built_track():
    """R49 ("replacing the fixed tube of 1.5 cm radius by a dynamic criterion taking into account the chi2").
    The straight-ish 20 GeV/c track of the first test with extra clusters on row 40.  The walking state there comes from the
    inner state (row 10) by Propagate alone, so its variances are those of the fit carried 30 rows: the test takes them from
    the pinned single Propagate step, builds the ellipse chi2 = dy^2 / (C00 + 0.01) + dz^2 / (C11 + 0.01) = 25 by hand and puts
    clusters 3 % inside and 3 % outside it on both axes and on the diagonal: inside -> adjacent and protected, outside ->
    untouched -- although every one of them lies well inside the fixed 1.5 cm tube, which alone would take them all."""
    rows = list(range(10, 70))
    tr = _helix_points(20.0, 1, 0.1, 0.3, -3.0, 20.0, rows)
    pts = [(r, p[1], p[2]) for r, p in zip(rows, tr)]
    ev, where = _event(pts)
    base = orc.run(ev, flags=True)
    st, cov = np.concatenate([[base.rf_x_in[0]], base.rf_par_in[0]]), base.rf_cov_in[0].copy()
    for r in range(11, 41):
        ok, st, cov = orc.propagate(st, cov, ROW_X[r], BZ, 0.98, fp64=False)
        assert ok
    ay, az = math.sqrt(25.0 * (cov[0] + 0.01)), math.sqrt(25.0 * (cov[2] + 0.01))     # half axes of the chi2 = 25 ellipse
    assert 0.5 < ay < 1.0 and 0.5 < az < 1.0                                          # far inside the 1.5 cm tube
    y40, z40 = st[1], st[2]
    d = math.sqrt(0.5)
    extra = [(40, y40 + 0.97 * ay, z40), (40, y40 + 1.03 * ay, z40), (40, y40, z40 - 0.97 * az), (40, y40, z40 - 1.03 * az),
             (40, y40 - 0.97 * d * ay, z40 + 0.97 * d * az), (40, y40 - 1.03 * d * ay, z40 + 1.03 * d * az)]
    ev, where = _event(pts + extra)
    p = orc.default_params()
    p.tube_chi2_max = 25.0
    res = orc.run(ev, p, flags=True)
    assert res.n_tracks == 1 and res.trk_ncl[0] == len(rows)
    e = where[len(rows):]
    assert [int(res.cf_flags[i]) for i in e] == [ADJ | PROT, RMB, ADJ | PROT, RMB, ADJ | PROT, RMB]
    assert np.all(res.cf_flags[where[:len(rows)]] == ATT | ADJ | PROT)                # the attached clusters always count (R35)
    res = orc.run(ev, flags=True)                                                      # fixed tube: all six are inside
    assert np.all(res.cf_flags[e] == ADJ | PROT)


def test_chi2_tube_equals_the_numpy_restatement_and_only_shrinks_the_tubes():
    ev = datagen.make_event(2, scale=0.03)
    p = orc.default_params()
    fixed = orc.run(ev, p, flags=True, merged=True)
    p.tube_chi2_max = 25.0
    res = orc.run(ev, p, flags=True, merged=True)
    f, owner, ry, rz = _flags_numpy(ev, res, p, rank=res.mt_rank)
    assert np.array_equal(owner, res.cf_owner) and np.array_equal(f, res.cf_flags)
    adj_f, adj_d = (fixed.cf_flags & ADJ) != 0, (res.cf_flags & ADJ) != 0
    assert not np.any(adj_d & ~adj_f) and adj_d.sum() < adj_f.sum()                  # a subset of the fixed tube
    assert np.array_equal((fixed.cf_flags & ATT) != 0, (res.cf_flags & ATT) != 0)
    noise = ev.truth_track < 0
    assert ((res.cf_flags & PROT) != 0)[noise].mean() < ((fixed.cf_flags & PROT) != 0)[noise].mean()     # fewer fake-protected
