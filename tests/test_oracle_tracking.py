"""Pins of the oracle's tracklet constructor (O4) and selector (O5) run as a whole.

BASELINE.json north_star checks 2 (noise-free high-pT helices fully found, every cluster attached),
3 (exact helix points -> generating parameters, through the whole pipeline), 4 (unit pulls within 5 %);
SURVEY.md 8(c) pins rows "O4 overall" (independence of processing order) and "O5 selector"
(<= 1 track per cluster; owner-by-priority == sequential greedy).
"""
import math

import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen
from paper_1910_12214_b200.datagen import GenConfig, Population
from tests.helpers import tri, truth_state_at_row

R = 152


def _single_sector_cfg(seed, n, pt_lo, pt_hi, sigma, phi_half_deg=8.0, eta_max=0.9):
    a = math.radians(10.0)
    w = math.radians(phi_half_deg)
    return GenConfig(seed, 1, [Population(0, n, pt_lo, pt_hi, phi_lo=a - w, phi_hi=a + w, eta_max=eta_max)],
                     sigma_y=sigma, sigma_z=sigma)


def test_noise_free_high_pt_helices_are_fully_found():
    """north_star check 2: one track per event, exact (unsmeared) crossings, pT >= 1 GeV/c."""
    n_found = 0
    for seed in range(1, 41):
        ev = datagen.generate(_single_sector_cfg(seed, 1, 1.0, 10.0, 0.0))
        if ev.n_clusters < 20:
            continue
        res = orc.run(ev)
        assert res.n_tracks == 1, seed
        assert np.array_equal(np.sort(res.trk_cl_index), np.arange(ev.n_clusters)), seed    # every cluster, nothing else
        assert res.trk_ncl[0] == ev.n_clusters
        n_found += 1
    assert n_found >= 35


def test_o4_operation_counters_of_one_full_length_track():
    """The O4 counters behind bench.py's algorithmic operation count, on a case the algorithm fixes:
    one noise-free track with a cluster on each of the n = 152 rows.  The end rows have no (up, down) pair, so the chain
    runs over rows 1..n-2: n-3 Propagate + Update in the chain fit, one Propagate + Search + Update for row n-1 going up,
    then n Propagates and n Updates going down with one Search (row 0): 2n-2, 2n-2, 2 Searches, 2 clusters inside the roads."""
    n_checked = 0
    for seed in range(1, 21):
        ev = datagen.generate(_single_sector_cfg(seed, 1, 1.0, 10.0, 0.0))
        if ev.n_clusters != R or np.any(np.diff(ev.row_offset.astype(np.int64)) != 1):
            continue
        res = orc.run(ev)
        assert res.o4_ops.tolist() == [2 * R - 2, 2 * R - 2, 2, 2], seed
        n_checked += 1
    assert n_checked >= 10


def test_exact_helix_through_the_whole_pipeline_fp64():
    """north_star check 3 through orcRun (fp64 arithmetic on fp32-rounded coordinates)."""
    checked = 0
    for seed in range(1, 25):
        ev = datagen.generate(_single_sector_cfg(seed, 1, 0.5, 10.0, 0.0, phi_half_deg=5.0))
        if ev.n_clusters < 100:
            continue
        res = orc.run(ev, fp64=True)
        assert res.n_tracks == 1
        x0 = float(ev.row_x[res.trk_first_row[0]])
        truth = truth_state_at_row(ev.trk_pt[0], ev.trk_phi0[0], ev.trk_eta[0], ev.trk_vz[0], ev.trk_h[0], ev.bz_tesla, 0,
                                   x0, n_sectors=1)
        fit = res.trk_par[0]
        # coordinates carry fp32 rounding (~4e-6 cm): positions to 1e-5 cm, angles to 1e-6, q/pT to 1e-4 relative
        assert abs(fit[0] - truth[0]) < 2e-5 and abs(fit[1] - truth[1]) < 5e-5
        assert abs(fit[2] - truth[2]) < 2e-6 and abs(fit[3] - truth[3]) < 2e-6
        assert abs(fit[4] - truth[4]) < 2e-4 * abs(truth[4]) + 2e-6
        checked += 1
    assert checked >= 10


@pytest.fixture(scope="module")
def pull_sample():
    pulls, chi2ndf = [], []
    for seed in range(100, 134):
        ev = datagen.generate(_single_sector_cfg(seed, 200, 0.5, 10.0, 0.1))
        res = orc.run(ev)
        cl_trk = ev.truth_track
        for k in range(res.n_tracks):
            idx = res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]]
            ids = cl_trk[idx]
            t = np.bincount(ids[ids >= 0]).argmax()
            if res.trk_ncl[k] < 60 or np.mean(ids == t) < 0.99:
                continue
            x0 = float(ev.row_x[res.trk_first_row[k]])
            truth = truth_state_at_row(ev.trk_pt[t], ev.trk_phi0[t], ev.trk_eta[t], ev.trk_vz[t], ev.trk_h[t],
                                       ev.bz_tesla, 0, x0, n_sectors=1)
            if truth is None:
                continue
            sig = np.sqrt(np.array([res.trk_cov[k][tri(i, i)] for i in range(5)]))
            pulls.append((res.trk_par[k] - truth) / sig)
            # ndf counts the tracklet's hits (the chi2 is the constructor's; R22)
            nh = res.tl_nhits[res.trk_tracklet[k]]
            chi2ndf.append(res.trk_chi2[k] / (2 * nh - 5))
    return np.array(pulls), np.array(chi2ndf)


def test_pull_widths_are_one_within_five_percent(pull_sample):
    """north_star check 4: pulls of smeared fits have unit width within 5 % (>= 5000 tracks, fp32 oracle)."""
    pulls, chi2ndf = pull_sample
    assert len(pulls) >= 5000
    # robust width (central 99.7 %) so that a handful of mis-assigned tracks do not decide the test
    for i in range(5):
        p = pulls[:, i]
        core = p[np.abs(p) < 4]
        assert len(core) > 0.995 * len(p)
        assert abs(core.std() - 1.0) < 0.05, (i, core.std())
        assert abs(core.mean()) < 0.05, (i, core.mean())
    assert abs(np.median(chi2ndf) - 1.0) < 0.05


def _remap_tracks(res, inv=None):
    out = set()
    for k in range(res.n_tracks):
        idx = res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]]
        if inv is not None:
            idx = inv[idx]
        out.add((tuple(int(i) for i in idx), tuple(np.asarray(res.trk_par[k], np.float32).tobytes())))
    return out


@pytest.mark.parametrize("idx,scale", [(1, 0.03), (2, 0.03)])
def test_results_do_not_depend_on_input_order(idx, scale):
    """Permuting the clusters inside every (sector,row) bucket permutes the result and nothing else:
    seeds are independent and every argmin is decided by values (ties aside, absent in smeared data)."""
    ev = datagen.make_event(idx, scale=scale)
    res = orc.run(ev)
    rng = np.random.default_rng(7)
    n = ev.n_clusters
    perm = np.arange(n)
    off = ev.row_offset.astype(np.int64)
    for b in range(len(off) - 1):
        perm[off[b]:off[b + 1]] = off[b] + rng.permutation(off[b + 1] - off[b])
    ev2 = datagen.event_from_arrays(ev.row_offset, ev.y[perm], ev.z[perm], ev.n_sectors, R)
    res2 = orc.run(ev2)
    # new index j holds old cluster perm[j]
    assert np.array_equal(np.where(res2.link_up >= 0, perm[np.maximum(res2.link_up, 0)], -1), res.link_up[perm])
    assert np.array_equal(np.sort(perm[res2.start_hits]), np.sort(res.start_hits))
    assert _remap_tracks(res2, perm) == _remap_tracks(res)


def _sequential_greedy(res, min_track_hits):
    """SURVEY.md 8(c) O5 'equivalent sequential formulation': sort tracklets by (-nhits, chi2, id); each in turn
    claims its still-unclaimed clusters."""
    acc = np.nonzero(res.tl_status == 2)[0]
    chi2 = res.tl_chi2.astype(np.float32)
    order = sorted(acc, key=lambda t: (-int(res.tl_nhits[t]), float(chi2[t]), int(t)))
    claimed = {}
    for t in order:
        for c in res.tl_rowhit[t]:
            if c >= 0 and c not in claimed:
                claimed[int(c)] = int(t)
    tracks = {}
    for t in acc:
        kept = [int(c) for c in res.tl_rowhit[t] if c >= 0 and claimed[int(c)] == t]
        if len(kept) >= min_track_hits:
            tracks[int(t)] = kept
    return tracks


@pytest.mark.parametrize("idx,scale", [(1, 0.05), (2, 0.05), (3, 0.04)])
def test_selector_equals_sequential_greedy_and_is_exclusive(idx, scale):
    ev = datagen.make_event(idx, scale=scale)
    p = orc.default_params()
    res = orc.run(ev, p)
    ref = _sequential_greedy(res, p.min_track_hits)
    assert list(res.trk_tracklet) == sorted(ref)                           # ascending tracklet id
    for k, t in enumerate(res.trk_tracklet):
        idx_k = res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]]
        assert list(idx_k) == ref[int(t)]                                  # ascending row = rowhit order
        assert res.trk_ncl[k] == len(idx_k)
        assert np.array_equal(res.trk_par[k], res.tl_par[t]) and res.trk_chi2[k] == res.tl_chi2[t]   # R22
    # exclusivity
    assert np.unique(res.trk_cl_index).size == res.trk_cl_index.size
    assert res.n_tracks > 10
    # tracklet bookkeeping: nhits == number of row hits; hits on first/last rows
    for t in np.nonzero(res.tl_status == 2)[0][:200]:
        rows = np.nonzero(res.tl_rowhit[t] >= 0)[0]
        assert len(rows) == res.tl_nhits[t] >= p.min_tracklet_hits
        assert rows[0] == res.tl_first_row[t] and rows[-1] == res.tl_last_row[t]


def test_tracking_efficiency_diagnostic_config1():
    """Not a pin (physics efficiency is 'parity unpinned'): a sanity floor that catches a broken constructor.
    Primaries with pT > 0.5 GeV/c and >= 100 clusters in one sector must nearly all be reconstructed."""
    ev = datagen.make_event(1, scale=0.1)
    res = orc.run(ev)
    bucket = np.repeat(np.arange(ev.n_sectors * R), np.diff(ev.row_offset.astype(np.int64)))
    sector = bucket // R
    key = ev.truth_track.astype(np.int64) * 64 + sector
    key = key[ev.truth_track >= 0]
    keys, counts = np.unique(key, return_counts=True)
    want = {int(k) for k, c in zip(keys, counts) if c >= 100 and ev.trk_pt[k // 64] > 0.5}
    found = set()
    for k in range(res.n_tracks):
        idx = res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]]
        ids = ev.truth_track[idx]
        ids = ids[ids >= 0]
        if len(ids) == 0:
            continue
        t = np.bincount(ids).argmax()
        if (ids == t).sum() >= 0.8 * len(idx) and len(idx) >= 70:
            found.add(int(t) * 64 + int(res.trk_sector[k]))
    assert len(want) > 100
    assert len(want & found) / len(want) > 0.97
