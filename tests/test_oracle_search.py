"""Decision-level pins of the oracle's Search (O4, reading R13) and of the control rules of the tracklet constructor
and the selector (R15 min_chain_hits, R16 max_row_gap, R18 min_tracklet_hits, R20 / R21
min_track_hits, R23 dead rows, step 5 "miss counting only below r0", step 6 "rows below the last snapshot").

Every expected value here is worked out by hand from the formula sheet (road = road_sigma * sqrt(C_mm + err2) clamped,
rectangular window, Euclidean nearest, ties to the lower index; the gap / threshold rules) on hand-built single-sector
events -- straight lines and one exact circle written with numpy apart from oracle/ -- and none comes from running
the oracle.  Each test names the line of oracle/tpc_oracle.cpp whose mutation it catches (checked by hand: see the
"catches" notes; the mutations were applied one at a time and the named test failed).
"""
import math

import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen
from paper_1910_12214_b200.datagen import default_row_x

R = 152
X = default_row_x().astype(np.float32).astype(np.float64)      # the row planes as the oracle sees them
DX = 160.0 / 151.0


# ---------------------------------------------------------------------------------------------------------------------
# (a), (b): one Search call on given clusters
# ---------------------------------------------------------------------------------------------------------------------
ROW = 30
YP, ZP = 1.0, 2.0                    # exactly representable road centre
C00, C10, C11 = 0.04, 0.02, 0.09     # three distinct values: a wrong covariance element changes a road


def _cov(c00=C00, c10=C10, c11=C11):
    c = np.zeros(15)
    c[0], c[1], c[2] = c00, c10, c11
    c[5], c[9], c[14] = 1e-4, 1e-4, 1e-2
    return c


def _search(pts, brute, params=None, cov=None, fp64=False):
    y = [p[0] for p in pts]
    z = [p[1] for p in pts]
    return orc.search([ROW] * len(pts), y, z, ROW, [X[ROW], YP, ZP, 0.1, 0.2, 0.5], _cov() if cov is None else cov,
                      X, params=params, brute=brute, fp64=fp64)


def _road(c, err2=0.01, sigma=4.0):
    """road_sigma * sqrt(C_mm + err2) in binary32, written apart from the oracle."""
    return float(np.float32(sigma) * np.sqrt(np.float32(c) + np.float32(err2)))


@pytest.mark.parametrize("brute", [False, True])
@pytest.mark.parametrize("fp64", [False, True])
def test_road_half_widths_come_from_c00_and_c11(brute, fp64):
    """ry = 4 sqrt(C00 + 0.01) = 0.8944, rz = 4 sqrt(C11 + 0.01) = 1.2649: a cluster 1e-4 inside is taken, 1e-4 outside
    is not, on both sides.  catches: oracle/tpc_oracle.cpp search(): st.C[0] -> st.C[1] or C[2] in ry, st.C[2] -> C[0]
    or C[1] in rz, err2_y <-> dropped, road_sigma dropped."""
    ry, rz = _road(C00), _road(C11)
    assert abs(ry - 0.894427) < 1e-5 and abs(rz - 1.264911) < 1e-5          # hand values
    for sg in (+1, -1):
        assert _search([(YP + sg * ry * (1 - 1e-4), ZP)], brute, fp64=fp64) == 0
        assert _search([(YP + sg * ry * (1 + 1e-4), ZP)], brute, fp64=fp64) == -1
        assert _search([(YP, ZP + sg * rz * (1 - 1e-4))], brute, fp64=fp64) == 0
        assert _search([(YP, ZP + sg * rz * (1 + 1e-4))], brute, fp64=fp64) == -1


@pytest.mark.parametrize("brute", [False, True])
def test_road_is_a_rectangle(brute):
    """R13: candidates have |dy| <= ry AND |dz| <= rz -- the corner of the rectangle is inside (an elliptical road
    (dy/ry)^2 + (dz/rz)^2 <= 1 would refuse it), and each coordinate is tested on its own."""
    ry, rz = _road(C00), _road(C11)
    assert _search([(YP + ry * 0.999, ZP - rz * 0.999)], brute) == 0
    assert _search([(YP + ry * 0.5, ZP + rz * 1.001)], brute) == -1
    assert _search([(YP - ry * 1.001, ZP + rz * 0.5)], brute) == -1


@pytest.mark.parametrize("brute", [False, True])
def test_road_clamps(brute):
    """Clamps to [road_min, road_max], NaN -> road_min.  With the defaults the raw width cannot fall below
    4 * sqrt(0.01) = 0.4, so road_min is raised to 0.5 to see it act.
    catches: the four clamp lines of search() (dropped, min <-> max, NaN falling through to road_max or to nothing)."""
    p = orc.default_params()
    p.road_min = 0.5
    cov = _cov(c00=0.0, c11=0.0)                                   # raw width 0.4 in both -> 0.5
    assert _search([(YP + 0.45, ZP)], brute, p, cov) == 0          # unclamped (0.4) would miss it
    assert _search([(YP + 0.4999, ZP)], brute, p, cov) == 0
    assert _search([(YP + 0.5001, ZP)], brute, p, cov) == -1
    assert _search([(YP, ZP - 0.4999)], brute, p, cov) == 0
    assert _search([(YP, ZP - 0.5001)], brute, p, cov) == -1
    cov = _cov(c00=1.0, c11=4.0)                                   # raw 4.02 and 8.01 -> 2.0
    q = orc.default_params()
    assert _search([(YP + 1.9998, ZP)], brute, q, cov) == 0
    assert _search([(YP + 2.0002, ZP)], brute, q, cov) == -1
    assert _search([(YP, ZP + 1.9998)], brute, q, cov) == 0
    assert _search([(YP, ZP + 2.0002)], brute, q, cov) == -1
    cov = _cov(c00=float("nan"), c11=float("nan"))                 # NaN -> road_min = 0.3
    assert _search([(YP + 0.2999, ZP)], brute, q, cov) == 0
    assert _search([(YP + 0.3001, ZP)], brute, q, cov) == -1
    assert _search([(YP, ZP + 0.2999)], brute, q, cov) == 0
    assert _search([(YP, ZP + 0.3001)], brute, q, cov) == -1
    cov = _cov(c00=-1.0, c11=-1.0)                                 # sqrt of a negative sum is NaN as well
    assert _search([(YP + 0.2999, ZP)], brute, q, cov) == 0
    assert _search([(YP + 0.3001, ZP)], brute, q, cov) == -1


@pytest.mark.parametrize("brute", [False, True])
def test_nearest_is_euclidean_and_ties_go_to_the_lower_index(brute):
    """Pick = min of (dy*dy + dz*dz, index).  Distances by hand:
    A = (0.28, 0): d2 0.0784;  B = (0.2, 0.2): d2 0.08          -> A  (max-norm or y alone would say B)
    A' = (0.3, 0): d2 0.09;    B                                 -> B  (the 1-norm 0.3 < 0.4 would say A')
    mirror points (+-0.125, 0) in either order -> index 0; in z likewise.
    catches: search(): d2 without dz*dz or without dy*dy, |dy|+|dz|, `c < best` -> `c > best`, `d2 < bestd` -> `>`."""
    A, B, A2 = (YP + 0.28, ZP), (YP + 0.2, ZP + 0.2), (YP + 0.3, ZP)
    assert _search([A, B], brute) == 0 and _search([B, A], brute) == 1
    assert _search([A2, B], brute) == 1 and _search([B, A2], brute) == 0
    Z1, Z2 = (YP, ZP + 0.28), (YP + 0.2, ZP - 0.2)                 # the same with y and z exchanged
    assert _search([Z1, Z2], brute) == 0 and _search([Z2, Z1], brute) == 1
    M1, M2 = (YP + 0.125, ZP), (YP - 0.125, ZP)                    # exact in binary32: a true tie
    assert _search([M1, M2], brute) == 0 and _search([M2, M1], brute) == 0
    N1, N2 = (YP, ZP + 0.25), (YP, ZP - 0.25)
    assert _search([N1, N2], brute) == 0 and _search([N2, N1], brute) == 0
    assert _search([M1, M2, (YP + 0.0625, ZP)], brute) == 2        # a nearer one later in the list still wins
    assert _search([], brute) == -1


def test_search_looks_only_at_the_asked_row():
    """Clusters of other rows at the road centre are not candidates."""
    rows = [ROW - 1, ROW, ROW + 1]
    y, z = [YP, YP + 0.5, YP], [ZP, ZP, ZP]
    for brute in (False, True):
        assert orc.search(rows, y, z, ROW, [X[ROW], YP, ZP, 0, 0, 0], _cov(), X, brute=brute) == 1
        assert orc.search(rows, y, z, ROW + 2, [X[ROW + 2], YP, ZP, 0, 0, 0], _cov(), X, brute=brute) == -1


# ---------------------------------------------------------------------------------------------------------------------
# (c), (d), (e): the control rules, through orcRun on hand-built events
# ---------------------------------------------------------------------------------------------------------------------
class Builder:
    """Clusters of one sector given as (row, y, z) in any order; input index = order inside the row = order added."""

    def __init__(self):
        self.pts = []

    def line(self, rows, y0=0.0, z0=10.0, ty=0.0, tz=0.0, xref=None, skip=()):
        xr = X[rows[0]] if xref is None else xref
        ids = {}
        for r in rows:
            if r in skip:
                continue
            ids[r] = self.add(r, y0 + ty * (X[r] - xr), z0 + tz * (X[r] - xr))
        return ids

    def add(self, r, y, z):
        self.pts.append((r, float(np.float32(y)), float(np.float32(z))))
        return len(self.pts) - 1

    def event(self, dead=()):
        order = sorted(range(len(self.pts)), key=lambda i: (self.pts[i][0], i))     # stable: by row, then as added
        self.index = {i: k for k, i in enumerate(order)}                            # builder id -> input index
        rows = np.array([self.pts[i][0] for i in order], np.int64)
        off = np.concatenate([[0], np.cumsum(np.bincount(rows, minlength=R))]).astype(np.uint32)
        rd = np.zeros(R, np.uint8)
        for r in dead:
            rd[r] = 1
        return datagen.event_from_arrays(off, [self.pts[i][1] for i in order], [self.pts[i][2] for i in order], 1, R,
                                         row_dead=rd)


def _rows_of(res, t):
    return [int(r) for r in np.nonzero(res.tl_rowhit[t] >= 0)[0]]


def _gap_event(k, dead=()):
    """A straight track (slopes 0.3, -0.2) on rows 10..40 and 41+k..80: k rows without a cluster above row 40."""
    b = Builder()
    b.line(list(range(10, 41)) + list(range(41 + k, 81)), y0=-3.0, z0=20.0, ty=0.3, tz=-0.2)
    return b.event(dead)


def test_gap_of_max_row_gap_rows_is_bridged_one_more_is_not():
    """R16: more than max_row_gap = 4 consecutive missed rows stop the extrapolation, in the up pass (step 3) and below
    r0 in the down pass (step 5).  By hand: the end clusters of a block have no (up, down) pair, so the lower block
    gives the chain rows 11..39 (start hit on row 11) and the upper block the chain rows 42+k..79 (start hit 42+k).
    k = 4: tracklet 0 misses rows 41..44 (4 <= 4), finds 45..80, stops after rows 81..85; going down it finds row 10 and
    stops after rows 9..5: rows 10..40 + 45..80 = 67 hits.  Tracklet 1 picks up row 80 going up and row 45 going down,
    misses the four rows 44..41, finds 40..10: the same 67 hits.  One track of 67 clusters.
    k = 5: the fifth miss stops both: tracklet 0 = rows 10..40 (31 hits), tracklet 1 = rows 46..80 (35 hits), two tracks.
    catches: construct(): `++miss > P.max_row_gap` -> `>=` (either pass), a hard-coded gap, misses not counted below r0."""
    ev = _gap_event(4)
    res = orc.run(ev)
    assert res.start_hits.tolist() == [1, 31 + 1]                 # clusters of rows 11 and 46 (= 42 + k)
    want = list(range(10, 41)) + list(range(45, 81))
    for t in (0, 1):
        assert _rows_of(res, t) == want and res.tl_nhits[t] == 67 and res.tl_status[t] == 2
        assert (res.tl_first_row[t], res.tl_last_row[t]) == (10, 80)
    assert res.n_tracks == 1 and res.trk_ncl[0] == 67
    assert np.array_equal(np.sort(res.trk_cl_index), np.arange(67))

    ev = _gap_event(5)
    res = orc.run(ev)
    assert res.start_hits.tolist() == [1, 31 + 1]                 # rows 11 and 47
    assert _rows_of(res, 0) == list(range(10, 41)) and res.tl_nhits[0] == 31
    assert _rows_of(res, 1) == list(range(46, 81)) and res.tl_nhits[1] == 35
    assert (res.tl_first_row[0], res.tl_last_row[0], res.tl_first_row[1], res.tl_last_row[1]) == (10, 40, 46, 80)
    assert res.n_tracks == 2 and res.trk_ncl.tolist() == [31, 35]

    p = orc.default_params()                                      # the parameter is what counts, not a constant 4
    p.max_row_gap = 5
    res = orc.run(ev, p)
    assert res.n_tracks == 1 and res.trk_ncl[0] == 66


def test_dead_rows_are_no_misses():
    """R23: five rows without clusters, one of them dead -> four misses -> bridged in both passes (the same event with
    the row alive is test ..._one_more_is_not, k = 5: not bridged).
    catches: construct(): `if (dead(r)) continue;` moved after the miss count / dropped, in step 3 and in step 5."""
    ev = _gap_event(5, dead=(43,))
    res = orc.run(ev)
    want = list(range(10, 41)) + list(range(46, 81))
    assert res.start_hits.tolist() == [1, 32]
    for t in (0, 1):
        assert _rows_of(res, t) == want and res.tl_nhits[t] == 66
    assert res.n_tracks == 1 and res.trk_ncl[0] == 66


def test_misses_inside_the_span_do_not_count_in_the_down_pass_and_a_hit_resets_the_count():
    """Step 5: going down, rows inside [r0, top] without a cluster are searched but are no misses; step 3: a found
    cluster resets the miss count.  Track on rows 10..30, 34..50, 54..70 (two gaps of three rows).  By hand: chains
    11..29, 35..49, 55..69; every tracklet bridges both gaps (3 <= 4 each; 6 in a row would not be) and holds all
    21 + 17 + 17 = 55 clusters, rows 10..70.
    catches: construct(): `miss = 0` after a found cluster dropped in step 3 (tracklet 0 would stop at row 50) or in step 5
    (tracklet 2 would stop at row 34); `else if (r < r0)` -> `else` (tracklet 0 would count 3 + 3 misses inside its span)."""
    b = Builder()
    b.line(list(range(10, 31)) + list(range(34, 51)) + list(range(54, 71)), y0=2.0, z0=-30.0, ty=-0.25, tz=0.4)
    res = orc.run(b.event())
    want = list(range(10, 31)) + list(range(34, 51)) + list(range(54, 71))
    assert res.start_hits.tolist() == [1, 21 + 1, 38 + 1]
    for t in range(3):
        assert _rows_of(res, t) == want and res.tl_nhits[t] == 55, t
        assert (res.tl_first_row[t], res.tl_last_row[t]) == (10, 70)
    assert res.n_tracks == 1 and res.trk_ncl[0] == 55


def test_search_is_centred_on_the_propagated_state():
    """Step 3: Propagate to the row, then Search around the predicted (y, z).  Straight track of slope 0.3 in y on rows
    10..40; four empty rows; on row 45 one cluster 0.25 cm above the line and one 0.15 cm below it: the lower one is
    nearer to the prediction and is taken (index order says the other).  A search around the position of the last hit
    (five rows * 0.3 * 1.06 = 1.6 cm away) finds neither.
    catches: construct() step 3: search before propagate; search(): centre st.y -> another element."""
    b = Builder()
    b.line(list(range(10, 41)), y0=-3.0, z0=20.0, ty=0.3, tz=-0.2)
    y45, z45 = -3.0 + 0.3 * (X[45] - X[10]), 20.0 - 0.2 * (X[45] - X[10])
    far = b.add(45, y45 + 0.25, z45)
    near = b.add(45, y45 - 0.15, z45)
    ev = b.event()
    res = orc.run(ev)
    assert res.tl_rowhit[0][45] == b.index[near] and b.index[near] > b.index[far]
    assert res.tl_nhits[0] == 32


@pytest.mark.parametrize("n_rows,status,nhits", [(4, 0, 2), (5, 1, 5), (9, 1, 9), (10, 2, 10), (11, 2, 11)])
def test_chain_and_tracklet_length_thresholds(n_rows, status, nhits):
    """R15 / R18 on a straight track of n consecutive rows starting at row 10.  By hand: its end clusters have no link
    pair, so the chain has n - 2 hits: n = 4 -> 2 < min_chain_hits = 3 -> status 0 (nhits = the chain's 2); n = 5 -> chain
    of 3, both ends picked up by the searches -> 5 hits < min_tracklet_hits = 10 -> status 1; n = 9 -> 9 -> status 1;
    n = 10 -> status 2 and a track of 10 clusters (min_track_hits = 10).
    catches: construct(): `nhits < P.min_chain_hits` -> `<=`; `snap_nh >= P.min_tracklet_hits` -> `>`;
    run(): `kept < P.min_track_hits` -> `<=`."""
    b = Builder()
    b.line(list(range(10, 10 + n_rows)), y0=1.0, z0=5.0, ty=0.1, tz=0.5)
    res = orc.run(b.event())
    assert res.start_hits.tolist() == [1]
    assert res.tl_status[0] == status and res.tl_nhits[0] == nhits
    if status:
        assert _rows_of(res, 0) == list(range(10, 10 + n_rows))
    assert res.n_tracks == (1 if status == 2 else 0)
    if status == 2:
        assert res.trk_ncl[0] == n_rows and res.trk_cl_index.tolist() == list(range(n_rows))


def test_thresholds_are_the_parameters():
    b = Builder()
    b.line(list(range(10, 20)), y0=1.0, z0=5.0, ty=0.1, tz=0.5)      # 10 clusters, chain of 8
    ev = b.event()
    p = orc.default_params()
    p.min_chain_hits = 9
    assert orc.run(ev, p).tl_status[0] == 0
    p = orc.default_params()
    p.min_tracklet_hits = 11
    res = orc.run(ev, p)
    assert res.tl_status[0] == 1 and res.n_tracks == 0
    p = orc.default_params()
    p.min_track_hits = 11
    res = orc.run(ev, p)
    assert res.tl_status[0] == 2 and res.n_tracks == 0
    p.min_tracklet_hits, p.min_track_hits = 5, 5
    b = Builder()
    b.line(list(range(10, 15)), y0=1.0, z0=5.0, ty=0.1, tz=0.5)
    res = orc.run(b.event(), p)
    assert res.tl_status[0] == 2 and res.n_tracks == 1 and res.trk_ncl[0] == 5


def _crossing_event(b_first_row):
    """Four straight tracks of one sector that share single clusters (the shared cluster is stored once):
      A  rows 0..39, y = 0, z = 10                                  (40 clusters)
      A2 rows 0..39, y, z = those of B on row 17                     (40 clusters)
      B  rows b_first_row..20, slopes (0.5, 1.0), through A on row 13 (S1) and through A2 on row 17 (S2)
      C  rows 16..25, slopes (-0.7, 1.0), through B's last cluster on row 20 (S3)          (10 clusters)
    Inside a row the clusters are stored in the order A, A2, B, C."""
    b = Builder()
    rowsA = list(range(0, 40))
    xb = X[13]
    yB = lambda r: 0.5 * (X[r] - xb)
    zB = lambda r: 10.0 + 1.0 * (X[r] - xb)
    ids = {"A": {}, "A2": {}, "B": {}, "C": {}}
    for r in range(0, 40):
        ids["A"][r] = b.add(r, 0.0, 10.0)
        ids["A2"][r] = b.add(r, yB(17), zB(17))
        if b_first_row <= r <= 20:
            if r == 13:
                ids["B"][r] = ids["A"][r]
            elif r == 17:
                ids["B"][r] = ids["A2"][r]
            else:
                ids["B"][r] = b.add(r, yB(r), zB(r))
        if 16 <= r <= 25:
            if r == 20:
                ids["C"][r] = ids["B"][r]
            else:
                ids["C"][r] = b.add(r, yB(20) - 0.7 * (X[r] - X[20]), zB(20) + 1.0 * (X[r] - X[20]))
    ev = b.event()
    return ev, {k: {r: b.index[i] for r, i in v.items()} for k, v in ids.items()}


def _track_sets(res):
    return [frozenset(int(c) for c in res.trk_cl_index[res.trk_cl_offset[k]:res.trk_cl_offset[k + 1]])
            for k in range(res.n_tracks)]


def test_min_track_hits_and_single_pass_ownership():
    """R19 (more hits first), R20 (a track needs min_track_hits = 10 kept clusters) and R21 (single pass: a tracklet
    that fails R20 still owns its clusters).  By hand, B on rows 10..20 (11 clusters): the shared clusters S1, S2 go to the
    40-hit tracklets of A and A2, B keeps 9 -> no track; C (10 hits) loses S3 to B (11 hits) and keeps 9 -> no track,
    although B itself is dropped: a second pass would hand S3 to C and make it a track of 10.  Tracks: A and A2, whole.
    With B on rows 9..20 (12 clusters) it keeps exactly 10 -> a third track (the boundary of R20), C still fails.
    The pair test of a shared cluster h: both lines through it give Dev = 0 for A / A2 (constant coordinates: the
    differences are exactly 0) -- the minimum, and on a tie the lower index, which is A's / A2's -- so S1, S2 stay in the
    chains of A, A2 and cut B's chain into pieces 11..12, 14..16, 18..19, of which only 14..16 reaches min_chain_hits.
    catches: run() O5: `kept < P.min_track_hits` -> `<=`; `better()`: nhits comparison reversed (S1 would go to B, A would
    have 39); a re-assignment of the clusters of failed tracklets (C would appear); owner test dropped in the keep loop."""
    ev, ids = _crossing_event(10)
    res = orc.run(ev)
    A, A2 = frozenset(ids["A"].values()), frozenset(ids["A2"].values())
    acc = [t for t in range(len(res.start_hits)) if res.tl_status[t] == 2]
    sets = {frozenset(int(c) for c in res.tl_rowhit[t] if c >= 0) for t in acc}
    assert sets == {A, A2, frozenset(ids["B"].values()), frozenset(ids["C"].values())}     # 40, 40, 11, 10 hits
    assert sorted(res.tl_nhits[acc].tolist()) == [10, 11, 40, 40]
    assert set(_track_sets(res)) == {A, A2}
    assert res.trk_ncl.tolist() == [40, 40]

    ev, ids = _crossing_event(9)
    res = orc.run(ev)
    A, A2 = frozenset(ids["A"].values()), frozenset(ids["A2"].values())
    Bkept = frozenset(ids["B"].values()) - {ids["B"][13], ids["B"][17]}
    assert len(Bkept) == 10
    assert set(_track_sets(res)) == {A, A2, Bkept}
    k = _track_sets(res).index(Bkept)
    assert (res.trk_first_row[k], res.trk_last_row[k], res.trk_ncl[k]) == (9, 20, 10)      # recomputed from the kept hits
    # R22: the parameters stay those of the tracklet (12 hits), not of the kept clusters
    assert res.tl_nhits[res.trk_tracklet[k]] == 12


def _circle_event(s_r0, k=-0.015, t=0.3, r_lo=19, r0=20, r_hi=60):
    """Exact circle through rows r_lo..r_hi: sin(phi) = s_r0 + k (x - x_r0); y = y0 + (cos phi_0 - cos phi) / k;
    z = z0 + t (phi - phi_0) / k  (written apart from the oracle; binary64, rounded once to binary32)."""
    b = Builder()
    c0 = math.sqrt(1 - s_r0 * s_r0)
    for r in range(r_lo, r_hi + 1):
        s = s_r0 + k * (X[r] - X[r0])
        b.add(r, 1.0 + (c0 - math.sqrt(1 - s * s)) / k, -40.0 + t * (math.asin(s) - math.asin(s_r0)) / k)
    return b.event()


def test_refused_propagate_in_the_down_pass_drops_the_rows_below_the_last_snapshot():
    """Step 5 / 6: "On break, hits on rows below the snapshot row are dropped".  A circle of curvature -0.015 / cm
    (pT = 0.1 GeV/c) with sin(phi) = 0.502 on row 20, falling with x, tracked with max_sinphi = 0.5.  By hand: the chain is
    rows 20..59 (row 19 only lends the start hit its down candidate); the chord of the first link has sin = 0.494 < 0.5, so
    the up pass runs and picks up row 60; coming down, the step from row 21 (sin 0.486) to row 20 needs sin 0.502 -> refused.
    Output = the snapshot of row 21: rows 21..60, 40 hits; the start hit itself is dropped from the row hits.
    With max_sinphi = 0.51 row 20 stays (41 hits) and the step to row 19 (sin 0.518) is refused; with 0.53 nothing is
    refused and rows 19..60 are all attached (42 hits).
    catches: construct(): `for (r < snap_row) rowhit[r] = -1` dropped (row 20 would stay, nhits 40 != 41 row hits);
    `if (!propagate(...)) break` -> continue in step 5; first_row taken from r0 instead of the snapshot."""
    ev = _circle_event(0.502)
    p = orc.default_params()
    p.max_sinphi = 0.5
    res = orc.run(ev, p)
    assert res.start_hits.tolist() == [1]                                   # the cluster of row 20
    assert _rows_of(res, 0) == list(range(21, 61))
    assert res.tl_nhits[0] == 40 and res.tl_status[0] == 2
    assert (res.tl_first_row[0], res.tl_last_row[0]) == (21, 60)
    assert res.tl_x[0] == pytest.approx(X[21], abs=1e-4)                    # the state is the snapshot's, at row 21
    assert res.n_tracks == 1 and res.trk_cl_index.tolist() == list(range(2, 42))
    assert abs(res.tl_par[0][2] - (0.502 - 0.015 * DX)) < 2e-4              # sin(phi) at row 21 of the circle
    assert abs(res.tl_par[0][4] - (-0.015 / (0.00299792458 * 0.5))) < 0.05  # q/pT = k / b = -10.007

    p.max_sinphi = 0.51
    res = orc.run(ev, p)
    assert _rows_of(res, 0) == list(range(20, 61)) and res.tl_nhits[0] == 41
    p.max_sinphi = 0.53
    res = orc.run(ev, p)
    assert _rows_of(res, 0) == list(range(19, 61)) and res.tl_nhits[0] == 42
    assert (res.tl_first_row[0], res.tl_last_row[0]) == (19, 60)


def test_refused_propagate_in_the_up_pass_ends_it_and_the_down_pass_still_runs():
    """Step 3: a refused Propagate ends the up extrapolation (no hit beyond), the tracklet is kept and goes down.
    The same circle rising with x, rows 19..45: sin(phi) = 0.30 on row 20, curvature +0.015 / cm -> 0.4907 on row 32 and
    0.5066 on row 33.  With max_sinphi = 0.5 the chain fit stops before row 33, the up extrapolation is refused at once,
    the down pass re-uses rows 32..20 and picks up row 19: rows 19..32 exactly, 14 hits.
    catches: construct() step 2 / 3: `if (!propagate(...)) break` -> the hit taken anyway; max_sinphi hard-coded."""
    s20, k = 0.30, 0.015
    s_of = lambda r: s20 + k * (X[r] - X[20])
    assert s_of(32) < 0.5 - 5e-3 and s_of(33) > 0.5 + 5e-3                  # the hand statement above, in numbers
    ev = _circle_event(s20, k=k, r_hi=45)
    p = orc.default_params()
    p.max_sinphi = 0.5
    res = orc.run(ev, p)
    t0 = 0
    assert _rows_of(res, t0) == list(range(19, 33)) and res.tl_nhits[t0] == 14
