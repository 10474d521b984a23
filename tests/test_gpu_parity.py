"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Sizes: the oracle finishes each case in seconds; the cases span many grid cells, several thread blocks
and ragged tails.  Full-size configs are covered by tests/test_gpu_full.py.
"""
import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen
from tests.parity import compare

pytestmark = pytest.mark.gpu

R = 152


def _tracker(ev, **par):
    from paper_1910_12214_b200 import tpc
    p = tpc.tpcDefaultParams()
    for k, v in par.items():
        setattr(p, k, v)
    return tpc.TpcTracker.from_event(ev, params=p)


def _oracle_params(**par):
    p = orc.default_params()
    for k, v in par.items():
        if hasattr(p, k):
            setattr(p, k, v)
    return p


def _run_both(ev, stages=True, **par):
    trk = _tracker(ev, **par)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, stages=stages)
    assert res.status.status == 0
    g = res.numpy()
    o = orc.run(ev, _oracle_params(**par))
    rep = compare(g, o, ev.n_rows, check_stages=stages)
    trk.close()
    return rep, res, o


@pytest.mark.parametrize("idx,scale", [(0, 1.0), (1, 0.1), (2, 0.1), (3, 0.06), (4, 0.02)])
def test_parity_configs_scaled(idx, scale):
    ev = datagen.make_event(idx, scale=scale)
    rep, res, o = _run_both(ev)
    assert o.n_tracks > 0
    print(ev.name, ev.n_clusters, "tracks", o.n_tracks, rep)


def test_parity_config1_full():
    """BASELINE.json configs[1] at full size (1.46 M clusters; the oracle needs ~2 s)."""
    ev = datagen.make_event(1)
    rep, res, o = _run_both(ev)
    assert o.n_tracks > 10000
    print(rep)


def test_parity_config2_full():
    ev = datagen.make_event(2)
    rep, res, o = _run_both(ev)
    print(rep)


def test_parity_dense_window_overflows_the_candidate_stash():
    """More than NF_STASH (12) down candidates per window: the re-enumeration path of the neighbour finder."""
    rng = np.random.default_rng(3)
    counts = np.zeros(R, np.int64)
    ys, zs = [], []
    for r in range(30, 60):
        k = 1500
        counts[r] = k
        ys.append(rng.uniform(-6, 6, k))
        zs.append(rng.uniform(-6, 6, k))      # ~10 clusters / cm^2 -> ~100 candidates per 3.2 x 3.2 cm window
    off = np.concatenate([[0], np.cumsum(counts)])
    ev = datagen.event_from_arrays(off, np.concatenate(ys), np.concatenate(zs), 1, R)
    rep, res, o = _run_both(ev)
    assert (o.link_up_raw >= 0).sum() > 1000


def test_parity_exact_ties_use_the_original_index():
    """Duplicated clusters (exact ties in Dev and in the search distance), shuffled input order."""
    ev0 = datagen.make_event(1, scale=0.02)
    rng = np.random.default_rng(11)
    counts = np.diff(ev0.row_offset.astype(np.int64))
    ys, zs, newc = [], [], []
    for b in range(len(counts)):
        lo, hi = ev0.row_offset[b], ev0.row_offset[b + 1]
        y = np.concatenate([ev0.y[lo:hi], ev0.y[lo:hi]])      # every cluster twice
        z = np.concatenate([ev0.z[lo:hi], ev0.z[lo:hi]])
        p = rng.permutation(len(y))
        ys.append(y[p])
        zs.append(z[p])
        newc.append(len(y))
    off = np.concatenate([[0], np.cumsum(newc)])
    ev = datagen.event_from_arrays(off, np.concatenate(ys), np.concatenate(zs), ev0.n_sectors, R)
    rep, res, o = _run_both(ev)
    assert o.n_tracks > 0


def test_parity_dead_rows():
    ev = datagen.make_event(0, dead_rows=(40, 97))
    rep, res, o = _run_both(ev)
    assert o.n_tracks > 50
    ev = datagen.make_event(1, scale=0.05, dead_rows=(1, 40, 41, 97, 150))
    _run_both(ev)


def test_parity_wide_selector_keys():
    """R27: the two-pass (wide) selector keys give the same tracks as the packed 64-bit key."""
    ev = datagen.make_event(2, scale=0.1)
    _run_both(ev, force_wide_keys=1)


def test_parity_other_parameters():
    ev = datagen.make_event(1, scale=0.05)
    _run_both(ev, road_sigma=3.0, max_row_gap=2, min_track_hits=20, min_tracklet_hits=15, link_dev2_max=0.3,
              clusters_per_cell=3.0)
    _run_both(ev, clusters_per_cell=0.25, cell_min=0.3)


def test_determinism_two_runs_identical_bytes():
    ev = datagen.make_event(3, scale=0.06)
    trk = _tracker(ev)
    off, y, z = trk.upload(ev)
    a = trk.run(off, y, z, stages=True).numpy()
    a = {k: v.copy() for k, v in a.items()}
    b = trk.run(off, y, z, stages=True).numpy()
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    trk.close()


def test_empty_and_tiny_inputs():
    from paper_1910_12214_b200 import tpc
    ev = datagen.event_from_arrays(np.zeros(R + 1, np.uint32), [], [], 1, R)
    trk = _tracker(ev)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, stages=True)
    assert res.status.status == 0 and res.n_tracks == 0 and res.status.n_start_hits == 0
    assert int(res.trk["trk_cl_offset"][0]) == 0
    trk.close()
    counts = np.zeros(R, np.int64)
    counts[10] = 1
    ev = datagen.event_from_arrays(np.concatenate([[0], np.cumsum(counts)]), [0.0], [0.0], 1, R)
    _run_both(ev)
    assert tpc.TPC_OK == 0


def test_capacity_overflow_is_reported_and_nothing_is_written_out_of_bounds():
    from paper_1910_12214_b200 import tpc
    ev = datagen.make_event(1, scale=0.1)
    trk = _tracker(ev)
    off, y, z = trk.upload(ev)
    full = trk.run(off, y, z)
    assert full.status.status == 0
    nt, nc, ns = full.n_tracks, full.n_track_clusters, int(full.status.n_start_hits)
    ref = {k: v.clone() for k, v in full.trk.items()}
    # tracks capacity too small: status CAPACITY, required sizes reported, the first cap tracks are intact
    res = trk.run(off, y, z, cap_tracks=nt // 2, grow=False)
    assert res.status.status == tpc.TPC_ERR_CAPACITY
    assert res.status.n_tracks == nt and res.status.n_track_clusters == nc
    assert np.array_equal(res.trk["trk_tracklet"].cpu().numpy(), ref["trk_tracklet"][:nt // 2].cpu().numpy())
    # cluster-index capacity too small
    res = trk.run(off, y, z, cap_track_clusters=nc // 3, grow=False)
    assert res.status.status == tpc.TPC_ERR_CAPACITY and res.status.n_track_clusters == nc
    # tracklet capacity too small: required cap_tracklets reported
    res = trk.run(off, y, z, cap_tracklets=ns // 2, grow=False)
    assert res.status.status == tpc.TPC_ERR_CAPACITY and res.status.n_start_hits == ns
    # and the automatic growth path recovers the full result
    res = trk.run(off, y, z, cap_tracklets=ns // 2, cap_tracks=nt // 2, cap_track_clusters=nc // 3)
    assert res.status.status == 0 and res.n_tracks == nt
    for k in ref:
        assert np.array_equal(res.trk[k].cpu().numpy(), ref[k].cpu().numpy()), k
    trk.close()


def test_bad_offsets_and_non_finite_input_are_reported():
    from paper_1910_12214_b200 import tpc
    ev = datagen.make_event(0)
    trk = _tracker(ev, validate_input=1)
    off, y, z = trk.upload(ev)
    bad = off.clone()
    bad[3] = bad[4] + 5            # off[4] < off[3]: not monotone
    with pytest.raises(tpc.TpcError) as e:
        trk.run(bad, y, z)
    assert e.value.code == tpc.TPC_ERR_UNSORTED_OFFSETS
    y2 = y.clone()
    y2[100] = float("nan")
    with pytest.raises(tpc.TpcError) as e:
        trk.run(off, y2, z)
    assert e.value.code == tpc.TPC_ERR_NONFINITE_INPUT
    res = trk.run(off, y, z)      # the handle is still usable
    assert res.status.status == 0 and res.n_tracks > 0
    trk.close()


def test_run_host_matches_device_path():
    ev = datagen.make_event(1, scale=0.1)
    trk = _tracker(ev)
    off, y, z = trk.upload(ev)
    dev = trk.run(off, y, z).numpy()
    st, host = trk.run_host(ev.row_offset, ev.y, ev.z)
    assert st.status == 0
    for k in host:
        assert np.array_equal(np.asarray(host[k]).view(np.int32) if host[k].dtype == np.uint32 else host[k], dev[k]), k
    trk.close()


@pytest.mark.parametrize("seed", list(range(12)))
def test_parity_fuzz_random_events_dead_rows_and_parameters(seed):
    """Seeded random small events: workload, size, dead rows, coarsened coordinates (many exact ties) and the
    parameters of Table P all vary; every stage must still be bit-identical to the oracle."""
    rng = np.random.default_rng(1000 + seed)
    idx = int(rng.integers(0, 5))
    scale = float({0: 0.6, 1: 0.04, 2: 0.05, 3: 0.03, 4: 0.008}[idx] * rng.uniform(0.5, 1.5))
    dead = tuple(int(r) for r in rng.choice(152, size=int(rng.integers(0, 6)), replace=False))
    ev = datagen.make_event(idx, scale=scale, seed=100 + seed, dead_rows=dead)
    if seed % 3 == 0:      # coordinates on a 1/8 cm lattice: exact ties in Dev and in the search distance
        ev = datagen.event_from_arrays(ev.row_offset, np.round(ev.y * 8) / 8, np.round(ev.z * 8) / 8, ev.n_sectors, R,
                                       row_dead=ev.row_dead)
    par = dict(road_sigma=float(rng.uniform(2.5, 6.0)), road_min=float(rng.uniform(0.1, 0.5)),
               road_max=float(rng.uniform(1.0, 3.0)), max_row_gap=int(rng.integers(1, 7)),
               min_chain_hits=int(rng.integers(2, 6)), min_tracklet_hits=int(rng.integers(5, 25)),
               min_track_hits=int(rng.integers(5, 25)), link_dev2_max=float(rng.uniform(0.1, 1.0)),
               area_y=float(rng.uniform(0.8, 2.0)), area_z=float(rng.uniform(0.8, 2.0)),
               max_sinphi=float(rng.uniform(0.8, 0.99)), clusters_per_cell=float(rng.uniform(0.2, 4.0)))
    rep, res, o = _run_both(ev, **par)
    assert len(o.start_hits) > 0


def test_submit_collect_pipeline_matches_run_host():
    """tpcSubmitHost / tpcCollectHost on two slots with different events in flight give, per event, exactly what the
    synchronous tpcRunHost gives; a too small capacity is reported, not overrun."""
    from paper_1910_12214_b200 import tpc
    import torch
    evs = [datagen.make_event(1, scale=0.05, seed=20 + i) for i in range(4)]
    trk = _tracker(evs[0])
    ref = []
    for ev in evs:
        st, out = trk.run_host(ev.row_offset, ev.y, ev.z)
        assert st.status == 0
        ref.append({k: v.copy() for k, v in out.items()})
    capK = max(len(r["trk_ncl"]) for r in ref) + 64
    capC = max(len(r["trk_cl_index"]) for r in ref) + 64

    def pin(a):
        return torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    ins = [(pin(ev.row_offset.astype(np.uint32)), pin(ev.y), pin(ev.z)) for ev in evs]
    trk.submit_host(0, *ins[0], capK, capC)
    for i in range(len(evs)):
        if i + 1 < len(evs):
            trk.submit_host((i + 1) % 2, *ins[i + 1], capK, capC)
        st, out = trk.collect_host(i % 2)
        assert st.status == 0 and st.n_tracks == len(ref[i]["trk_ncl"])
        for k in ref[i]:
            assert np.array_equal(out[k], ref[i][k]), (i, k)
    # capacity too small for the tracks: reported, the valid prefix only is exposed
    trk.submit_host(0, *ins[0], 8, capC)
    st, out = trk.collect_host(0)
    assert st.status == tpc.TPC_ERR_CAPACITY and len(out["trk_ncl"]) == 8
    # a slot must be collected before it is reused
    trk.submit_host(1, *ins[1], capK, capC)
    with pytest.raises(tpc.TpcError):
        trk.submit_host(1, *ins[2], capK, capC)
    st, out = trk.collect_host(1)
    assert st.status == 0
    trk.close()


def test_shared_denominator_division_is_bit_identical_to_the_ieee_division():
    """R0 for the one place where the kernels do not write `a / S`: the Kalman update's six quotients by one reciprocal
    (csrc/tpc_kalman.cuh).  2^26 threads x 48 operand pairs over the whole domain of the shared form, zeros of both signs,
    exact quotients, the edge of the domain and overflowing quotients included: no bit pattern may differ."""
    from paper_1910_12214_b200 import tpc
    ev = datagen.make_event(0, scale=0.05)
    trk = tpc.TpcTracker.from_event(ev)
    tested = 0
    for seed in (1, 2, 3):
        n, bad = tpc.tpcSelfTestDivision(trk.handle, 1 << 26, seed)
        assert bad == 0, (seed, bad, n)
        tested += n
    trk.close()
    assert tested == 3 * 48 * (1 << 26)


def test_parity_on_the_hand_built_events_of_the_control_rule_pins():
    """The hand-built events of tests/test_oracle_search.py (gaps of max_row_gap and one more, dead rows inside a gap, gaps
    inside the span, two candidates in a road, chains and tracklets around the length thresholds, four crossing lines that
    share single clusters, a Propagate refused in the down pass and in the up pass): the oracle's answers there are worked
    out by hand, and the CUDA path must give the same, bit for bit -- these are the cases that drive the gap instance of the
    span pass, the rows-below-the-snapshot rule and the single-pass ownership of the selector."""
    from tests import test_oracle_search as S
    cases = [(S._gap_event(4), {}), (S._gap_event(5), {}), (S._gap_event(5), {"max_row_gap": 5}), (S._gap_event(5, dead=(43,)), {}),
             (S._crossing_event(10)[0], {}), (S._crossing_event(9)[0], {}),
             (S._circle_event(0.502), {"max_sinphi": 0.5}), (S._circle_event(0.502), {"max_sinphi": 0.51}),
             (S._circle_event(0.502), {"max_sinphi": 0.53}), (S._circle_event(0.30, k=0.015, r_hi=45), {"max_sinphi": 0.5})]
    b = S.Builder()
    b.line(list(range(10, 31)) + list(range(34, 51)) + list(range(54, 71)), y0=2.0, z0=-30.0, ty=-0.25, tz=0.4)
    cases.append((b.event(), {}))
    for n in (4, 5, 9, 10, 11):
        b = S.Builder()
        b.line(list(range(10, 10 + n)), y0=1.0, z0=5.0, ty=0.1, tz=0.5)
        cases.append((b.event(), {}))
        cases.append((b.event(), {"min_chain_hits": 4, "min_tracklet_hits": 5, "min_track_hits": 5}))
    for ev, par in cases:
        rep, res, o = _run_both(ev, **par)
        assert rep["exact"] and rep["tl_exact"], (par, rep)


def test_parity_when_a_bucket_has_more_cells_than_the_shared_histogram_holds():
    """a1 `gridBuild` keeps the cell histogram of a bucket in shared memory up to 24 576 cells; with `clusters_per_cell` =
    0.003 the ~117 clusters of a config-0 bucket get ~39 000 cells, and the same passes run on the bucket's slice of the
    global cell table with the arrival ranks in `rank`.  The grid never decides a result (R3): everything stays bit-exact."""
    ev = datagen.make_event(0)
    trk = _tracker(ev, clusters_per_cell=0.003)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, stages=True)
    assert res.status.status == 0
    assert res.status.n_cells > 24576 * 100                  # most of the 152 buckets are above the shared-memory limit
    rep = compare(res.numpy(), orc.run(ev), ev.n_rows)
    trk.close()
    assert rep["exact"] and rep["tl_exact"]
