"""-m gpu: the optional a7 segment merger (through the C ABI) against the oracle's O7: links, heads and the chi2 of
every link are bit-identical (integer outputs exactly; the chi2 is fp32 computed in the same order on both sides)."""
import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen

pytestmark = pytest.mark.gpu


def _both(ev, **par):
    from paper_1910_12214_b200 import tpc
    p = tpc.tpcDefaultParams()
    po = orc.default_params()
    for k, v in par.items():
        setattr(p, k, v)
        setattr(po, k, v)
    trk = tpc.TpcTracker.from_event(ev, params=p)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, merge=True)
    assert res.status.status == 0
    g = res.numpy()
    trk.close()
    o = orc.run(ev, po, merge=True)
    assert g["trk_mg_next"].shape[0] == o.n_tracks
    assert np.array_equal(g["trk_cl_index"].view(np.uint32), o.trk_cl_index)
    assert np.array_equal(g["trk_rf_status"], o.rf_status)
    assert np.array_equal(g["trk_mg_next"], o.mg_next)
    assert np.array_equal(g["trk_mg_prev"], o.mg_prev)
    assert np.array_equal(g["trk_mg_head"], o.mg_head)
    assert np.array_equal(g["trk_mg_chi2"], o.mg_chi2.astype(np.float32))
    return g, o, res


@pytest.mark.parametrize("idx,scale", [(1, 0.1), (2, 0.1), (3, 0.05), (4, 0.015)])
def test_merge_parity(idx, scale):
    ev = datagen.make_event(idx, scale=scale)
    g, o, res = _both(ev)
    assert (o.mg_next >= 0).sum() > 20
    cross = o.trk_sector[o.mg_next >= 0] != o.trk_sector[o.mg_next[o.mg_next >= 0]]
    assert cross.any()                                         # links across sector borders are exercised
    assert res.status.merge_ms >= 0.0


def test_merge_parity_single_sector_with_a_band_of_removed_rows_and_other_cuts():
    ev = datagen.make_event(0)
    off = ev.row_offset.astype(np.int64)
    keep = np.ones(ev.n_clusters, bool)
    keep[off[70]:off[80]] = False
    counts = np.diff(off)
    counts[70:80] = 0
    ev2 = datagen.event_from_arrays(np.concatenate([[0], np.cumsum(counts)]), ev.y[keep], ev.z[keep], 1, ev.n_rows)
    g, o, _ = _both(ev2)
    assert (o.mg_next >= 0).sum() > 50                         # the cut tracks are rejoined
    g, o, _ = _both(ev2, merge_max_row_gap=12, merge_chi2_max=8.0)
    g, o, _ = _both(datagen.make_event(1, scale=0.05), merge_back_rows=0, merge_max_row_gap=80, merge_chi2_max=200.0)


def test_merge_needs_the_refit_outputs():
    from paper_1910_12214_b200 import tpc
    ev = datagen.make_event(0)
    trk = tpc.TpcTracker.from_event(ev)
    off, y, z = trk.upload(ev)
    trk._ensure(ev.n_clusters, 4096, 4096, ev.n_clusters, False, False, True)     # merger outputs without refit outputs
    cl = tpc.tpcClusters(ev.n_clusters, off.data_ptr(), None, y.data_ptr(), z.data_ptr(), None)
    tr = tpc.tpcTracks()
    tr.cap_tracks, tr.cap_track_clusters = 4096, ev.n_clusters
    for k, v in trk._out.items():
        setattr(tr, k, v.data_ptr())
    with pytest.raises(tpc.TpcError):
        tpc.tpcRun(trk.handle, cl, tr, 4096, trk._ws.data_ptr(), trk._ws.numel(), 0)
    trk.close()
