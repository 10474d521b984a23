"""-m gpu: the optional a10 pairs of looper legs (through the C ABI) against the oracle's O10: partners and the chi2 of
every pair are bit-identical (integer outputs exactly; the chi2 is fp32 computed in the same order on both sides)."""
import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen

pytestmark = pytest.mark.gpu


def _both(ev, merge=False, **par):
    from paper_1910_12214_b200 import tpc
    p = tpc.tpcDefaultParams()
    po = orc.default_params()
    for k, v in par.items():
        setattr(p, k, v)
        setattr(po, k, v)
    trk = tpc.TpcTracker.from_event(ev, params=p)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, legs=True, merge=merge)
    assert res.status.status == 0
    g = res.numpy()
    trk.close()
    o = orc.run(ev, po, legs=True, merge=merge)
    assert g["trk_leg_partner"].shape[0] == o.n_tracks
    assert np.array_equal(g["trk_cl_index"].view(np.uint32), o.trk_cl_index)
    assert np.array_equal(g["trk_rf_status"], o.rf_status)
    assert np.array_equal(g["trk_leg_partner"], o.lg_partner)
    assert np.array_equal(g["trk_leg_chi2"], o.lg_chi2.astype(np.float32))
    if merge:
        assert np.array_equal(g["trk_mg_next"], o.mg_next) and np.array_equal(g["trk_mg_head"], o.mg_head)
    return g, o, res


@pytest.mark.parametrize("idx,scale,least", [(2, 0.15, 300), (1, 0.1, 0), (3, 0.05, 0), (4, 0.012, 0)])
def test_legs_parity(idx, scale, least):
    ev = datagen.make_event(idx, scale=scale)
    g, o, res = _both(ev)
    assert (o.lg_partner >= 0).sum() >= least
    assert res.status.legs_ms >= 0.0


def test_legs_parity_with_other_cuts_dead_rows_and_the_merger_beside_it():
    ev = datagen.make_event(2, scale=0.1, dead_rows=(30, 31, 90))
    g, o, _ = _both(ev, merge=True)
    assert (o.lg_partner >= 0).sum() > 100
    _both(ev, leg_min_sinphi=0.2, leg_chi2_max=500.0, leg_max_sectors=8, leg_max_row_diff=40, leg_max_centre_dist=60.0)
    _both(ev, leg_max_centre_dist=0.7)
    _both(ev, leg_min_sinphi=0.8, leg_chi2_max=5.0, leg_max_sectors=0, leg_max_row_diff=0)
    _both(ev, leg_max_sectors=2, max_sinphi=0.9)


def test_legs_parity_single_sector_geometry():
    ev = datagen.make_event(0)                     # one sector: only d = 0 is compared
    g, o, _ = _both(ev, leg_min_sinphi=0.05, leg_chi2_max=1e6, leg_max_row_diff=151, leg_max_centre_dist=1e4)
    assert g["trk_leg_partner"].shape[0] > 100


def test_legs_need_the_refit_outputs_and_both_pointers():
    from paper_1910_12214_b200 import tpc
    ev = datagen.make_event(0)
    trk = tpc.TpcTracker.from_event(ev)
    off, y, z = trk.upload(ev)
    cl = tpc.tpcClusters(ev.n_clusters, off.data_ptr(), None, y.data_ptr(), z.data_ptr(), None)
    for refit, drop in ((False, None), (True, "trk_leg_chi2")):
        trk._ensure(ev.n_clusters, 4096, 4096, ev.n_clusters, False, refit, False, False, False, True)
        tr = tpc.tpcTracks()
        tr.cap_tracks, tr.cap_track_clusters = 4096, ev.n_clusters
        for k, v in trk._out.items():
            if k != drop:
                setattr(tr, k, v.data_ptr())
        with pytest.raises(tpc.TpcError):
            tpc.tpcRun(trk.handle, cl, tr, 4096, trk._ws.data_ptr(), trk._ws.numel(), 0)
    p = tpc.tpcDefaultParams()
    p.leg_max_sectors = 9
    with pytest.raises(tpc.TpcError):
        tpc.TpcTracker.from_event(ev, params=p)
    trk.close()


@pytest.mark.parametrize("seed", list(range(8)))
def test_fuzz_all_optional_stages_together(seed):
    """Seeded random small events and parameters with the refit, the merger, the leg pairs and the cluster flags all
    switched on in one tpcRun: every optional output must still be bit-identical to the oracle's."""
    from paper_1910_12214_b200 import tpc
    rng = np.random.default_rng(4000 + seed)
    idx = int(rng.integers(1, 5))
    scale = float({1: 0.04, 2: 0.06, 3: 0.03, 4: 0.008}[idx] * rng.uniform(0.6, 1.4))
    dead = tuple(int(r) for r in rng.choice(152, size=int(rng.integers(0, 5)), replace=False))
    ev = datagen.make_event(idx, scale=scale, seed=300 + seed, dead_rows=dead)
    par = dict(max_sinphi=float(rng.uniform(0.85, 0.99)), min_track_hits=int(rng.integers(6, 20)),
               merge_max_row_gap=int(rng.integers(5, 80)), merge_back_rows=int(rng.integers(0, 10)),
               merge_chi2_max=float(rng.uniform(5.0, 200.0)), tube_radius=float(rng.uniform(0.5, 3.0)),
               inv_pt_protect=float(rng.uniform(2.0, 30.0)), leg_min_sinphi=float(rng.uniform(0.1, 0.9)),
               leg_chi2_max=float(rng.uniform(5.0, 300.0)), leg_max_sectors=int(rng.integers(0, 9)),
               leg_max_row_diff=int(rng.integers(0, 40)), leg_max_centre_dist=float(rng.uniform(0.5, 50.0)))
    p, po = tpc.tpcDefaultParams(), orc.default_params()
    for k, v in par.items():
        setattr(p, k, v)
        setattr(po, k, v)
    trk = tpc.TpcTracker.from_event(ev, params=p)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, legs=True, merge=True, flags=True)
    assert res.status.status == 0
    g = res.numpy()
    trk.close()
    o = orc.run(ev, po, legs=True, merge=True, flags=True)
    assert np.array_equal(g["trk_cl_index"].view(np.uint32), o.trk_cl_index)
    assert np.array_equal(g["trk_rf_status"], o.rf_status)
    assert np.array_equal(g["trk_rf_par_out"], o.rf_par_out.T.astype(np.float32))
    assert np.array_equal(g["trk_leg_partner"], o.lg_partner) and np.array_equal(g["trk_leg_chi2"], o.lg_chi2.astype(np.float32))
    assert np.array_equal(g["trk_mg_next"], o.mg_next) and np.array_equal(g["trk_mg_prev"], o.mg_prev)
    assert np.array_equal(g["trk_mg_head"], o.mg_head) and np.array_equal(g["trk_mg_chi2"], o.mg_chi2.astype(np.float32))
    assert np.array_equal(g["cl_flags"], o.cf_flags) and np.array_equal(g["cl_owner"], o.cf_owner)
    assert np.array_equal(g["cl_res_y"], o.cf_res_y.astype(np.float32)) and np.array_equal(g["cl_res_z"], o.cf_res_z.astype(np.float32))
