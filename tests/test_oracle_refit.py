"""Pins of the oracle's O6 refit (NEXT-2 of SURVEY.md 8(f); DESIGN.md section 3 "O6", readings R28..R30).

The refit is a composition of Propagate and Update, each pinned on its own in tests/test_oracle_kalman.py
(closed-form asin helix, finite differences, numpy matrix Kalman update).  What is pinned here is the
composition itself -- which clusters enter, in which order, with which priors, and which state comes out
at which end -- against things it does not compute itself: the closed-form helix (exact points are
recovered at BOTH ends), numpy.polyfit, unit pulls at both ends, and bookkeeping invariants of the whole
pipeline.  All CPU (-m "not gpu").
"""
import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen
from tests.helpers import KAPPA, helix_step_closed_form, tri

BZ = 0.5
ROW_X = (85.0 + np.arange(152) * (160.0 / 151.0)).astype(np.float32).astype(np.float64)


def _exact(pt, s0, t, charge, rows, y0=2.0, z0=-30.0):
    """Exact helix points on the given rows (closed form), starting at rows[0]."""
    st0 = np.array([ROW_X[rows[0]], y0, z0, s0, t, charge / pt])
    return np.array([helix_step_closed_form(st0, ROW_X[r] - ROW_X[rows[0]], BZ) for r in rows])


@pytest.mark.parametrize("pt,s0,t,charge", [(0.3, 0.2, 0.5, 1), (1.0, -0.3, -0.8, -1), (5.0, 0.1, 0.2, 1),
                                            (10.0, 0.0, 1.0, -1)])
def test_refit_recovers_exact_helix_at_both_ends(pt, s0, t, charge):
    """Exact helix points (with gaps in the row sequence) -> the generating state at the first AND at the last
    cluster to 1e-5 relative in binary64, chi2 = 0."""
    rows = np.array([r for r in range(5, 120) if r % 7 != 3])          # ragged: missing rows
    pts = _exact(pt, s0, t, charge, rows)
    assert np.all(np.abs(pts[:, 3]) < 0.9)
    ok, inner, outer = orc.refit_points(rows, pts[:, 1], pts[:, 2], ROW_X, BZ, fp64=True)
    assert ok
    for got, truth in ((inner, pts[0]), (outer, pts[-1])):
        assert got[0] == pytest.approx(truth[0], abs=1e-12)            # x of the reference plane
        floor = np.array([1.0, 1.0, 1.0, 1.0, abs(truth[5])])
        assert np.all(np.abs(got[1:6] - truth[1:]) <= 1e-5 * np.maximum(np.abs(truth[1:]), floor)), (got[:6], truth)
    assert inner[21] < 1e-8
    # the up pass starts from the prior q/pT = 0 +- sqrt(init_var_q): exact data leave exactly that pull in its chi2
    assert outer[21] == pytest.approx((charge / pt) ** 2 / 100.0, rel=2e-2, abs=1e-6)
    ok32, in32, out32 = orc.refit_points(rows, pts[:, 1], pts[:, 2], ROW_X, BZ, fp64=False)
    assert ok32
    assert np.all(np.abs(in32[1:5] - pts[0][1:5]) <= 1e-4 * np.maximum(np.abs(pts[0][1:5]), 1.0))
    assert np.all(np.abs(out32[1:5] - pts[-1][1:5]) <= 1e-4 * np.maximum(np.abs(pts[-1][1:5]), 1.0))


def test_refit_equals_least_squares_parabola_at_small_angles():
    """Textbook special case: small angles, diffuse priors -> ordinary least squares (numpy.polyfit), at both ends."""
    rng = np.random.default_rng(5)
    rows = np.arange(20, 90)
    pts = _exact(8.0, 0.01, 0.05, 1.0, rows, y0=0.5, z0=3.0)
    ys = pts[:, 1] + rng.normal(0, 0.1, len(rows))
    zs = pts[:, 2] + rng.normal(0, 0.1, len(rows))
    ok, inner, outer = orc.refit_points(rows, ys, zs, ROW_X, BZ, fp64=True)
    assert ok
    xs = ROW_X[rows]
    for got, xref in ((inner, xs[0]), (outer, xs[-1])):
        u = xs - xref
        cy = np.polyfit(u, ys, 2)
        cz = np.polyfit(u, zs, 1)
        sig = np.sqrt(np.array([got[6 + tri(i, i)] for i in range(5)]))
        # the down pass starts from a 1 cm^2 prior, the up pass from the first cluster itself: both ~ plain least squares
        assert abs(got[1] - cy[2]) < 5e-2 * sig[0]
        assert abs(got[3] - cy[1]) < 5e-2 * sig[2]
        assert abs(got[5] * KAPPA * BZ - 2 * cy[0]) < 5e-2 * sig[4] * KAPPA * BZ
        assert abs(got[2] - cz[1]) < 5e-2 * sig[1]
        assert abs(got[4] - cz[0]) < 5e-2 * sig[3]
    # the same data in both passes: the two ends describe the same helix
    fwd = helix_step_closed_form(inner[:6], xs[-1] - xs[0], BZ)
    sig_o = np.sqrt(np.array([outer[6 + tri(i, i)] for i in range(5)]))
    assert np.all(np.abs(fwd[1:] - outer[1:6]) < 0.1 * sig_o)


def test_refit_pulls_have_unit_width_at_both_ends():
    """Pulls (estimate - truth) / sigma of all five parameters, inner and outer state, 4000 smeared tracks."""
    rng = np.random.default_rng(77)
    pulls_in, pulls_out, chi2ndf = [], [], []
    n_tracks = 4000
    while len(pulls_in) < n_tracks:
        pt = np.exp(rng.uniform(np.log(0.5), np.log(10.0)))
        charge = rng.choice([-1.0, 1.0])
        r0 = int(rng.integers(0, 40))
        rows = np.arange(r0, r0 + int(rng.integers(40, 100)))
        rows = rows[rng.random(len(rows)) > 0.1]                         # 10 % of the clusters lost to other tracks
        if len(rows) < 20:
            continue
        pts = _exact(pt, rng.uniform(-0.3, 0.3), rng.uniform(-0.8, 0.8), charge, rows, y0=rng.uniform(-5, 5),
                     z0=rng.uniform(-100, 100))
        if np.any(np.abs(pts[:, 3]) > 0.8):
            continue
        ys = pts[:, 1] + rng.normal(0, 0.1, len(rows))
        zs = pts[:, 2] + rng.normal(0, 0.1, len(rows))
        ok, inner, outer = orc.refit_points(rows, ys, zs, ROW_X, BZ, fp64=False)      # the parity precision
        assert ok
        for got, truth, dst in ((inner, pts[0], pulls_in), (outer, pts[-1], pulls_out)):
            sig = np.sqrt(np.array([got[6 + tri(i, i)] for i in range(5)]))
            dst.append((got[1:6] - truth[1:]) / sig)
        chi2ndf.append(inner[21] / (2 * len(rows) - 5))
    for pulls in (np.array(pulls_in), np.array(pulls_out)):
        for i in range(5):
            p = pulls[:, i]
            core = p[np.abs(p) < 4]
            assert len(core) > 0.995 * len(p)
            assert abs(core.std() - 1.0) < 0.05, (i, core.std())
            assert abs(core.mean()) < 0.06, (i, core.mean())
    assert abs(np.mean(chi2ndf) - 1.0) < 0.05


def test_refit_rejects_what_it_cannot_fit():
    ok, _, _ = orc.refit_points(np.array([3]), np.array([0.0]), np.array([0.0]), ROW_X, BZ)
    assert not ok                                                         # fewer than two clusters
    ok, _, _ = orc.refit_points(np.array([5, 4]), np.zeros(2), np.zeros(2), ROW_X, BZ)
    assert not ok                                                         # rows must ascend
    ok, _, _ = orc.refit_points(np.array([10, 11, 12]), np.array([0.0, 30.0, 60.0]), np.zeros(3), ROW_X, BZ)
    assert not ok                                                         # |sin phi| beyond max_sinphi


def test_refit_in_the_pipeline_bookkeeping_and_quality():
    """orc.run(refit=True): one refit per track, reference planes on the first / last kept cluster, the O1..O5 results
    untouched, chi2/ndf ~ 1 on smeared config-0 data, and equal to refit_points on the track's own clusters."""
    ev = datagen.make_event(0)
    base = orc.run(ev)
    res = orc.run(ev, refit=True)
    assert res.n_tracks == base.n_tracks > 100
    assert np.array_equal(res.trk_cl_index, base.trk_cl_index) and np.array_equal(res.trk_par, base.trk_par)
    assert np.all(res.rf_status == 1)
    row_x = np.asarray(ev.row_x, np.float32).astype(np.float64)
    assert np.array_equal(res.rf_x_in, row_x[res.trk_first_row]) and np.array_equal(res.rf_x_out, row_x[res.trk_last_row])
    ndf = 2 * res.trk_ncl - 5
    assert abs(np.median(res.rf_chi2 / ndf) - 1.0) < 0.1
    rowof = np.repeat(np.arange(ev.n_rows * ev.n_sectors), np.diff(ev.row_offset.astype(np.int64))) % ev.n_rows
    for k in range(0, res.n_tracks, 17):
        idx = res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]]
        ok, inner, outer = orc.refit_points(rowof[idx], ev.y[idx].astype(np.float64), ev.z[idx].astype(np.float64),
                                            row_x, ev.bz_tesla, fp64=False)
        assert ok
        assert np.array_equal(inner[1:6], res.rf_par_in[k]) and np.array_equal(inner[6:21], res.rf_cov_in[k])
        assert np.array_equal(outer[1:6], res.rf_par_out[k]) and inner[21] == res.rf_chi2[k]
