"""-m gpu: the optional a11 merged tracks and leg labels (through the C ABI) against the oracle's O12, and the a8 cluster
flags with the leg labels in (secondary legs do not protect, PAPER.md L83 / L86): everything bit-exact."""
import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen

pytestmark = pytest.mark.gpu


def _both(ev, flags=True, **par):
    from paper_1910_12214_b200 import tpc
    p = tpc.tpcDefaultParams()
    po = orc.default_params()
    for k, v in par.items():
        setattr(p, k, v)
        if hasattr(po, k):
            setattr(po, k, v)
    trk = tpc.TpcTracker.from_event(ev, params=p)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, merged=True, flags=flags, pos=flags)
    assert res.status.status == 0
    g = res.numpy()
    trk.close()
    o = orc.run(ev, po, merged=True, flags=flags)
    assert np.array_equal(g["trk_cl_index"].view(np.uint32), o.trk_cl_index)
    assert np.array_equal(g["trk_mg_next"], o.mg_next) and np.array_equal(g["trk_leg_partner"], o.lg_partner)
    assert np.array_equal(g["trk_mt_id"], o.mt_id)
    assert np.array_equal(g["trk_mt_rank"], o.mt_rank)
    assert np.array_equal(g["mt_cl_offset"].view(np.uint32), o.mt_cl_offset)
    assert np.array_equal(g["mt_cl_index"].view(np.uint32), o.mt_cl_index)
    if flags:
        assert np.array_equal(g["cl_owner"], o.cf_owner)
        assert np.array_equal(g["cl_flags"], o.cf_flags)
        assert np.array_equal(g["cl_res_y"], o.cf_res_y.astype(np.float32))
        assert np.array_equal(g["cl_res_code"].view(np.uint32), o.cf_res_code)
    return g, o, res


@pytest.mark.parametrize("idx,scale", [(2, 1.0), (2, 0.1), (1, 0.1), (3, 0.05), (0, 1.0)])
def test_merged_tracks_and_flags_parity(idx, scale):
    ev = datagen.make_event(idx, scale=scale)
    g, o, res = _both(ev)
    if idx == 2:
        assert (o.mt_rank == 1).sum() > 20                      # two-leg merged tracks are exercised
        sec = o.mt_rank[np.repeat(np.arange(o.n_tracks), o.trk_ncl)] == 1
        f = o.cf_flags[o.trk_cl_index[sec]]
        assert ((f & 8) != 0).mean() > 0.8                      # most clusters of secondary legs go with strategy A
    assert res.status.merged_ms >= 0.0


def test_merged_tracks_parity_dead_rows_and_other_cuts():
    ev = datagen.make_event(2, scale=0.2, dead_rows=(30, 31, 90))
    _both(ev)
    _both(ev, leg_chi2_max=400.0, leg_max_centre_dist=30.0, merge_chi2_max=200.0, merge_max_row_gap=80)
    _both(ev, flags=False)
    _both(ev, tube_chi2_max=25.0)                       # chi2 tube together with the leg labels


def test_merged_outputs_need_the_merger_and_the_leg_pairs():
    from paper_1910_12214_b200 import tpc
    ev = datagen.make_event(0)
    trk = tpc.TpcTracker.from_event(ev)
    off, y, z = trk.upload(ev)
    trk._ensure(ev.n_clusters, 4096, 4096, ev.n_clusters, False, True, True, False, False, False, False, True)   # no leg outputs
    cl = tpc.tpcClusters(ev.n_clusters, off.data_ptr(), None, y.data_ptr(), z.data_ptr(), None)
    tr = tpc.tpcTracks()
    tr.cap_tracks, tr.cap_track_clusters = 4096, ev.n_clusters
    for k, v in trk._out.items():
        setattr(tr, k, v.data_ptr())
    with pytest.raises(tpc.TpcError):
        tpc.tpcRun(trk.handle, cl, tr, 4096, trk._ws.data_ptr(), trk._ws.numel(), 0)
    trk.close()
