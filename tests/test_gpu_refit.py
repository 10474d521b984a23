"""-m gpu: the optional a6 refit (through the C ABI) against the oracle's O6, element by element.

The bar is the north_star's: parameters 1e-4 relative, covariances 1e-3 relative; with R0 honoured on both
sides the results are in fact bit-identical, and that is what is asserted (the tolerances are head-room).
"""
import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen
from tests.parity import compare

pytestmark = pytest.mark.gpu


def _run(ev, **kw):
    from paper_1910_12214_b200 import tpc
    trk = tpc.TpcTracker.from_event(ev)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, refit=True, **kw)
    assert res.status.status == 0
    g = res.numpy()
    trk.close()
    return res, g


def _check(ev, g, o):
    nt = o.n_tracks
    assert g["trk_rf_status"].shape[0] == nt
    assert np.array_equal(g["trk_rf_status"], o.rf_status)
    pairs = [("trk_rf_x_in", o.rf_x_in), ("trk_rf_chi2", o.rf_chi2), ("trk_rf_x_out", o.rf_x_out),
             ("trk_rf_par_in", o.rf_par_in.T), ("trk_rf_cov_in", o.rf_cov_in.T), ("trk_rf_par_out", o.rf_par_out.T),
             ("trk_rf_cov_out", o.rf_cov_out.T)]
    worst = 0.0
    for name, ref in pairs:
        a, b = g[name].astype(np.float64), np.asarray(ref, np.float64)
        assert a.shape == b.shape, name
        tol = 1e-3 if "cov" in name else 1e-4
        err = np.abs(a - b) / np.maximum(np.abs(b), 1e-6)
        assert np.all(err <= tol), (name, err.max())
        worst = max(worst, float(err.max()) if err.size else 0.0)
        assert np.array_equal(g[name], np.asarray(ref, np.float32)), name      # in fact bit-identical
    return worst


@pytest.mark.parametrize("idx,scale", [(0, 1.0), (1, 0.1), (2, 0.1), (4, 0.02)])
def test_refit_parity(idx, scale):
    ev = datagen.make_event(idx, scale=scale)
    res, g = _run(ev)
    o = orc.run(ev, refit=True)
    assert compare(g, o, ev.n_rows, check_stages=False)        # a1..a5 untouched by the refit
    assert o.n_tracks > 0 and int(o.rf_status.sum()) > 0.95 * o.n_tracks
    _check(ev, g, o)
    assert res.status.stage_ms[7] >= 0.0


def test_refit_parity_dead_rows_and_duplicates():
    ev0 = datagen.make_event(1, scale=0.03)
    dead = np.zeros(ev0.n_rows, np.uint8)
    dead[[40, 97]] = 1
    off = ev0.row_offset.astype(np.int64).copy()
    keep = np.ones(ev0.n_clusters, bool)
    for s in range(ev0.n_sectors):
        for r in (40, 97):
            b = s * ev0.n_rows + r
            keep[off[b]:off[b + 1]] = False
    counts = np.diff(off)
    bucket = np.repeat(np.arange(len(counts)), counts)
    newc = np.bincount(bucket[keep], minlength=len(counts))
    y, z = ev0.y[keep], ev0.z[keep]
    # every cluster twice: exact ties everywhere (R6), zero-length steps never occur (rows differ)
    o2 = np.concatenate([[0], np.cumsum(2 * newc)])
    yy, zz = [], []
    o1 = np.concatenate([[0], np.cumsum(newc)])
    for b in range(len(newc)):
        yy += [y[o1[b]:o1[b + 1]]] * 2
        zz += [z[o1[b]:o1[b + 1]]] * 2
    ev = datagen.event_from_arrays(o2, np.concatenate(yy), np.concatenate(zz), ev0.n_sectors, ev0.n_rows, row_dead=dead)
    res, g = _run(ev)
    o = orc.run(ev, refit=True)
    assert o.n_tracks > 0
    _check(ev, g, o)


def test_refit_outputs_are_all_or_none_and_capacity_overflow_skips_the_refit():
    from paper_1910_12214_b200 import tpc
    ev = datagen.make_event(0)
    trk = tpc.TpcTracker.from_event(ev)
    off, y, z = trk.upload(ev)
    full = trk.run(off, y, z, refit=True)
    n = full.n_tracks
    # too few track slots: status CAPACITY, the refit kernel does not run on truncated lists (nothing out of bounds)
    res = trk.run(off, y, z, refit=True, cap_tracks=max(n // 2, 1), grow=False)
    assert res.status.status == tpc.TPC_ERR_CAPACITY
    # all-or-none: a partial set of refit pointers is an argument error
    trk._ensure(ev.n_clusters, 4096, 4096, ev.n_clusters, False, True)
    cl = tpc.tpcClusters(ev.n_clusters, off.data_ptr(), None, y.data_ptr(), z.data_ptr(), None)
    tr = tpc.tpcTracks()
    tr.cap_tracks, tr.cap_track_clusters = 4096, ev.n_clusters
    for k, v in trk._out.items():
        setattr(tr, k, v.data_ptr())
    tr.trk_rf_chi2 = None
    with pytest.raises(tpc.TpcError):
        tpc.tpcRun(trk.handle, cl, tr, 4096, trk._ws.data_ptr(), trk._ws.numel(), 0)
    trk.close()
