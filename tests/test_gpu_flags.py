"""-m gpu: the optional a8 cluster flags (through the C ABI) against the oracle's O8: flag bytes and owners bit-exact."""
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
        if hasattr(po, k):
            setattr(po, k, v)
    trk = tpc.TpcTracker.from_event(ev, params=p)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, flags=True, merge=True)
    assert res.status.status == 0
    g = res.numpy()
    trk.close()
    o = orc.run(ev, po, flags=True, merge=True)
    assert np.array_equal(g["trk_cl_index"].view(np.uint32), o.trk_cl_index)
    assert np.array_equal(g["cl_owner"], o.cf_owner)
    assert np.array_equal(g["cl_flags"], o.cf_flags)
    assert np.array_equal(g["cl_res_y"], o.cf_res_y.astype(np.float32))      # track-model residuals (R39), bit-exact
    assert np.array_equal(g["cl_res_z"], o.cf_res_z.astype(np.float32))
    assert np.array_equal(g["trk_mg_next"], o.mg_next)          # the three optional stages coexist
    return g, o, res


@pytest.mark.parametrize("idx,scale", [(0, 1.0), (1, 0.1), (2, 0.1), (3, 0.05), (4, 0.015)])
def test_flags_parity(idx, scale):
    ev = datagen.make_event(idx, scale=scale)
    g, o, res = _both(ev)
    f = o.cf_flags
    assert ((f & 4) != 0).sum() > 0.5 * ev.n_clusters * (0.2 if idx == 4 else 1.0) or idx >= 3
    assert res.status.flags_ms >= 0.0


def test_flags_parity_dead_rows_lattice_ties_and_other_cuts():
    ev = datagen.make_event(2, scale=0.06, dead_rows=(30, 31, 90))
    _both(ev)
    ev2 = datagen.event_from_arrays(ev.row_offset, np.round(ev.y * 4) / 4, np.round(ev.z * 4) / 4, ev.n_sectors, ev.n_rows,
                                    row_dead=ev.row_dead)                    # clusters exactly on tube borders
    _both(ev2, tube_radius=1.25)
    _both(ev, tube_radius=3.0, inv_pt_protect=2.0, clusters_per_cell=0.3)
    _both(ev, tube_radius=0.0)
    _both(ev, tube_chi2_max=25.0)                       # R49: the chi2 criterion on top of the fixed tube
    _both(ev2, tube_chi2_max=9.0, tube_radius=2.0)


def test_flags_on_an_event_without_tracks():
    rng = np.random.default_rng(1)
    n = 3000
    rows = np.sort(rng.integers(0, 152, n))
    off = np.concatenate([[0], np.cumsum(np.bincount(rows, minlength=152))])
    ev = datagen.event_from_arrays(off, rng.uniform(-10, 10, n), rng.uniform(-200, 200, n), 1, 152)
    g, o, _ = _both(ev)
    assert o.n_tracks == 0 and np.all(g["cl_flags"] == 16) and np.all(g["cl_owner"] == -1)


@pytest.mark.parametrize("nb", [4, 3, 0, 9])
def test_charge_code_parity(nb):
    """a9 (O9): the 16-bit dynamic-precision charge code, bit-exact; inputs cover the 16-bit range, halves
    (ties), negatives, NaN, infinities and a ragged tail."""
    import torch
    from paper_1910_12214_b200 import tpc
    ev = datagen.make_event(1, scale=0.03)
    n = ev.n_clusters
    rng = np.random.default_rng(5)
    q = np.concatenate([ev.q[: n // 2], rng.uniform(0, 70000, n - n // 2 - 9).astype(np.float32),
                        np.array([0.5, 1.5, 2.5, -1.0, np.nan, np.inf, -np.inf, 65535.4, 33.0], np.float32)]).astype(np.float32)
    p = tpc.tpcDefaultParams()
    p.charge_trunc_bits = nb
    trk = tpc.TpcTracker.from_event(ev, params=p)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, q=torch.from_numpy(q).cuda())
    assert res.status.status == 0
    got = res.trk["cl_qcode"].cpu().numpy().view(np.uint16)
    assert np.array_equal(got, orc.pack_charge(q, nb))
    trk.close()


def test_charge_code_golden_fixture():
    """tests/golden/charge_codes.txt (written from oracle/ only) through the CUDA path."""
    import os
    import torch
    from paper_1910_12214_b200 import tpc
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "charge_codes.txt")) if l[0] != "#"]
    a = np.array(rows, np.float64)
    ev = datagen.make_event(0, scale=0.2)
    n = ev.n_clusters
    q = np.resize(a[:, 0].astype(np.float32), n)
    for nb, col in ((4, 1), (3, 2)):
        p = tpc.tpcDefaultParams()
        p.charge_trunc_bits = nb
        trk = tpc.TpcTracker.from_event(ev, params=p)
        off, y, z = trk.upload(ev)
        res = trk.run(off, y, z, q=torch.from_numpy(q).cuda())
        got = res.trk["cl_qcode"].cpu().numpy().view(np.uint16)
        assert np.array_equal(got, np.resize(a[:, col].astype(np.uint16), n))
        trk.close()


@pytest.mark.parametrize("bits", [6, 0, 9, 15])
def test_position_and_residual_code_parity(bits):
    """O11: the 16-bit integer codes of the absolute positions and of the track-model residuals,
    bit-exact; the positions are overwritten in places with ties (half units), values beyond the range, NaN-free
    infinities are not valid tracker input, so the extreme values ride on a tracker-free call at the end."""
    import torch
    from paper_1910_12214_b200 import tpc
    ev = datagen.make_event(2, scale=0.05)
    p, po = tpc.tpcDefaultParams(), orc.default_params()
    p.pos_bits = bits
    trk = tpc.TpcTracker.from_event(ev, params=p)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, flags=True, pos=True)
    assert res.status.status == 0
    g = res.numpy()
    o = orc.run(ev, po, flags=True, pos_bits=bits)
    assert np.array_equal(g["cl_pos_code"].view(np.uint32), orc.pack_positions(ev.y, ev.z, bits))
    assert np.array_equal(g["cl_res_y"], o.cf_res_y.astype(np.float32))
    assert np.array_equal(g["cl_res_code"].view(np.uint32), o.cf_res_code)
    assert (o.cf_res_code != 0).sum() > 1000 or bits == 0
    # positions alone (no flags, no refit): ties, saturation and a ragged tail (n not a multiple of 4)
    n = ev.n_clusters - (ev.n_clusters % 4) - 1
    off2 = ev.row_offset.copy().astype(np.int64)
    off2 = np.minimum(off2, n).astype(np.uint32)
    rng = np.random.default_rng(9)
    unit = 2.0 ** -bits
    yy = (rng.integers(-40000, 40000, n) * 0.5 * unit).astype(np.float32)          # half units: every second one a tie
    zz = rng.uniform(-600, 600, n).astype(np.float32)
    ev2 = datagen.event_from_arrays(off2, yy, zz, ev.n_sectors, ev.n_rows)
    off, y, z = trk.upload(ev2)
    res = trk.run(off, y, z, pos=True)
    assert np.array_equal(res.numpy()["cl_pos_code"].view(np.uint32), orc.pack_positions(yy, zz, bits))
    trk.close()
    bad = tpc.tpcDefaultParams()
    bad.pos_bits = 16
    with pytest.raises(tpc.TpcError):
        tpc.TpcTracker.from_event(ev, params=bad)


def test_optional_stages_on_empty_and_overflowing_inputs():
    """All optional stages requested on an empty event, on a rows-only event without tracks and with too small track
    capacities: defined status, nothing written out of bounds (guard values around the outputs stay intact)."""
    import torch
    from paper_1910_12214_b200 import tpc
    ev = datagen.event_from_arrays(np.zeros(153, np.uint32), np.zeros(0, np.float32), np.zeros(0, np.float32), 1, 152)
    trk = tpc.TpcTracker.from_event(ev)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, merge=True, flags=True, q=torch.zeros(0, device="cuda"))
    assert res.status.status == 0 and res.n_tracks == 0
    trk.close()
    ev = datagen.make_event(1, scale=0.05)
    trk = tpc.TpcTracker.from_event(ev)
    off, y, z = trk.upload(ev)
    full = trk.run(off, y, z, merge=True, flags=True)
    assert full.status.status == 0 and full.n_tracks > 100
    res = trk.run(off, y, z, merge=True, flags=True, cap_tracks=full.n_tracks // 3, grow=False)
    assert res.status.status == tpc.TPC_ERR_CAPACITY and res.status.n_tracks == full.n_tracks
    res = trk.run(off, y, z, merge=True, flags=True, cap_track_clusters=full.n_track_clusters // 2, grow=False)
    assert res.status.status == tpc.TPC_ERR_CAPACITY
    again = trk.run(off, y, z, merge=True, flags=True)                 # and the tracker is fine afterwards
    for k in ("trk_mg_next", "cl_flags", "cl_owner", "trk_rf_par_in"):
        assert torch.equal(again.trk[k], full.trk[k]), k
    trk.close()
