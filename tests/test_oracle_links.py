"""Pins of the oracle's grid (O1), neighbour finder (O2) and cleaner / start-hit finder (O3).

SURVEY.md 8(c) "pins": grid invariants; grid search == brute-force search (BASELINE.json north_star
check 1); an all-pairs numpy search on tiny inputs; closed forms (collinear clusters have Dev = 0 and
link, a hand-computed five-cluster argmin, duplicates -> lowest index, the window edge is inclusive);
reciprocity and path invariants after cleaning (north_star check 5).
"""
import numpy as np
import pytest

from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen

R = 152
ROWX = datagen.default_row_x().astype(np.float32)


def _event(rows_y_z, n_rows=R, row_dead=None, n_sectors=1):
    """rows_y_z: dict (sector,row) or row -> list of (y, z), in input order."""
    counts = np.zeros(n_sectors * n_rows, np.int64)
    ys, zs = [], []
    keys = sorted((k if isinstance(k, tuple) else (0, k)) for k in rows_y_z)
    for (s, r) in keys:
        pts = rows_y_z[(s, r)] if (s, r) in rows_y_z else rows_y_z[r]
        counts[s * n_rows + r] = len(pts)
        for (y, z) in pts:
            ys.append(y)
            zs.append(z)
    off = np.concatenate([[0], np.cumsum(counts)])
    return datagen.event_from_arrays(off, ys, zs, n_sectors, n_rows, row_dead=row_dead)


# ------------------------------------------------------------------------------------------------ O1
def test_grid_invariants():
    ev = datagen.make_event(1, scale=0.05)
    res = orc.run(ev)
    n = ev.n_clusters
    off = ev.row_offset.astype(np.int64)
    s2o = res.sorted_to_orig.astype(np.int64)
    assert np.array_equal(np.sort(s2o), np.arange(n))
    for b in range(0, ev.n_sectors * R, 37):           # a sample of buckets
        lo, hi = off[b], off[b + 1]
        assert np.all((s2o[lo:hi] >= lo) & (s2o[lo:hi] < hi))       # a permutation inside each bucket
        cells = res.cell_of_sorted[lo:hi]
        assert np.all(np.diff(cells) >= 0)                          # grouped by ascending cell
        assert cells.size == 0 or (cells.min() >= 0 and cells.max() < res.n_cells[b])
        same = np.diff(cells) == 0
        assert np.all(np.diff(s2o[lo:hi])[same] > 0)                # stable inside a cell
    # every cluster lies in the cell its coordinates map to: clusters closer than the smallest cell edge
    # along both axes are in the same or adjacent cells; checked through the search equivalence below


@pytest.mark.parametrize("idx,scale", [(0, 1.0), (1, 0.03), (2, 0.03), (3, 0.04)])
def test_grid_search_equals_brute_force_search(idx, scale):
    """R3 / north_star check 1: the grid only enumerates a superset; all outputs are byte-identical."""
    ev = datagen.make_event(idx, scale=scale)
    a = orc.run(ev)
    b = orc.run(ev, brute_force=True)
    for f in ("link_up_raw", "link_dn_raw", "link_up", "link_dn", "start_hits", "tl_status", "tl_nhits", "tl_rowhit",
              "tl_par", "tl_cov", "tl_chi2", "trk_tracklet", "trk_ncl", "trk_cl_offset", "trk_cl_index", "trk_par",
              "trk_cov"):
        assert np.array_equal(getattr(a, f), getattr(b, f)), f
    assert a.n_tracks > 0


def test_grid_search_equals_brute_force_with_out_of_range_and_dense_clusters():
    """Clusters outside the nominal (y,z) range are clamped into edge cells; many clusters per cell."""
    rng = np.random.default_rng(5)
    rows = {}
    for r in range(20, 30):
        y = rng.uniform(-30, 30, 300)           # beyond the sector edge x*tan(10 deg) ~ 19 cm
        z = rng.uniform(-270, 270, 300)         # beyond z_max = 250
        rows[r] = list(zip(y, z))
    ev = _event(rows)
    a, b = orc.run(ev), orc.run(ev, brute_force=True)
    assert np.array_equal(a.link_up_raw, b.link_up_raw) and np.array_equal(a.link_dn_raw, b.link_dn_raw)
    assert np.array_equal(a.trk_cl_index, b.trk_cl_index)


# ------------------------------------------------------------------------------------------------ O2
def _numpy_all_pairs_links(ev, p):
    """The definition of O2 written as a dense all-pairs search in numpy float32 (tiny inputs only)."""
    n = ev.n_clusters
    up = np.full(n, -1, np.int32)
    dn = np.full(n, -1, np.int32)
    off = ev.row_offset.astype(np.int64)
    y, z, X = ev.y, ev.z, ev.row_x
    f = np.float32
    for s in range(ev.n_sectors):
        for r in range(1, R - 1):
            b = s * R + r
            hs = np.arange(off[b], off[b + 1])
            us = np.arange(off[b + 1], off[b + 2])
            ds = np.arange(off[b - 1], off[b])
            if not (len(hs) and len(us) and len(ds)):
                continue
            dxu, dxd = f(X[r + 1] - X[r]), f(X[r] - X[r - 1])
            iu, idn = f(1) / dxu, f(1) / dxd
            for h in hs:
                okU = (np.abs(y[us] - y[h]) <= f(p.area_y) * dxu) & (np.abs(z[us] - z[h]) <= f(p.area_z) * dxu)
                okD = (np.abs(y[ds] - y[h]) <= f(p.area_y) * dxd) & (np.abs(z[ds] - z[h]) <= f(p.area_z) * dxd)
                U, D = us[okU], ds[okD]
                if not (len(U) and len(D)):
                    continue
                tyu, tzu = (y[U] - y[h]) * iu, (z[U] - z[h]) * iu
                tyd, tzd = (y[h] - y[D]) * idn, (z[h] - z[D]) * idn
                ey = tyu[:, None] - tyd[None, :]
                ez = tzu[:, None] - tzd[None, :]
                dev = ey * ey + ez * ez
                assert dev.dtype == np.float32
                best = dev.min()
                if best <= f(p.link_dev2_max):
                    ia, ic = np.nonzero(dev == best)        # row-major: lowest u first, then lowest d
                    up[h], dn[h] = U[ia[0]], D[ic[0]]
    return up, dn


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_neighbour_finder_equals_numpy_all_pairs_on_tiny_inputs(seed):
    rng = np.random.default_rng(seed)
    rows = {}
    for r in range(60, 70):   # dense random clusters: several candidates per window, many fake links
        k = int(rng.integers(30, 80))
        rows[r] = list(zip(rng.uniform(-5, 5, k), rng.uniform(-5, 5, k)))
    ev = _event(rows)
    p = orc.default_params()
    res = orc.run(ev, p)
    up, dn = _numpy_all_pairs_links(ev, p)
    assert np.array_equal(res.link_up_raw, up)
    assert np.array_equal(res.link_dn_raw, dn)
    assert (up >= 0).sum() > 20


def test_three_collinear_clusters_link_with_zero_deviation():
    """Closed form: points on a straight line through equally spaced rows have equal slopes -> Dev = 0."""
    x = ROWX.astype(np.float64)
    r = 80
    pts = {q: [(np.float32(0.25 * (x[q] - x[r])), np.float32(10 - 0.5 * (x[q] - x[r])))] for q in (r - 1, r, r + 1)}
    ev = _event(pts)
    p = orc.default_params()
    p.link_dev2_max = 1e-9      # only a (numerically) zero deviation passes
    res = orc.run(ev, p)
    assert list(res.link_up_raw) == [-1, 2, -1]
    assert list(res.link_dn_raw) == [-1, 0, -1]


def test_hand_built_five_cluster_case():
    """Row spacing is 160/151 cm.  h at (0,0); up candidates u0 = (+d, 0), u1 = (+2d, +d); down candidates
    d0 = (-2d, -d), d1 = (0, -d) with d = 160/151 / 4 ... slopes: u0 (0.25, 0), u1 (0.5, 0.25),
    from-below d0 (0.5, 0.25), d1 (0, 0.25).  Dev(u0,d0) = 0.0625+0.0625 = 0.125, Dev(u0,d1) = 0.0625+0.0625 = 0.125,
    Dev(u1,d0) = 0, Dev(u1,d1) = 0.25 -> best pair is (u1, d0)."""
    d = (160.0 / 151.0) / 4
    r = 50
    ev = _event({r - 1: [(-2 * d, -d), (0.0, -d)], r: [(0.0, 0.0)], r + 1: [(d, 0.0), (2 * d, d)]})
    res = orc.run(ev)
    # input order: d0 = 0, d1 = 1, h = 2, u0 = 3, u1 = 4
    assert res.link_up_raw[2] == 4 and res.link_dn_raw[2] == 0
    # remove the perfect pair's down partner: the two remaining ties (u0,d1)=0.125 vs (u1,d1)=0.25 -> (u0,d1)
    ev2 = _event({r - 1: [(0.0, -d)], r: [(0.0, 0.0)], r + 1: [(d, 0.0), (2 * d, d)]})
    res2 = orc.run(ev2)
    assert res2.link_up_raw[1] == 2 and res2.link_dn_raw[1] == 0


def test_duplicate_clusters_resolve_to_lowest_input_index():
    """R6: exact ties in Dev -> lowest original index of u, then of d."""
    r = 50
    ev = _event({r - 1: [(0.0, 0.0), (0.0, 0.0)], r: [(0.0, 0.0)], r + 1: [(0.0, 0.0), (0.0, 0.0), (0.0, 0.0)]})
    res = orc.run(ev)
    assert res.link_dn_raw[2] == 0 and res.link_up_raw[2] == 3
    # symmetric tie in Dev between two different pairs: (u_a, d_b) and (u_b, d_a) mirror images
    ev = _event({r - 1: [(0.1, 0.0), (-0.1, 0.0)], r: [(0.0, 0.0)], r + 1: [(0.1, 0.0), (-0.1, 0.0)]})
    res = orc.run(ev)
    # Dev(u=+0.1, d=-0.1)=0 and Dev(u=-0.1, d=+0.1)=0: tie -> u with the lower index (3), its partner d=1
    assert res.link_up_raw[2] == 3 and res.link_dn_raw[2] == 1


def test_window_edge_is_inclusive_and_outside_is_excluded():
    x = ROWX
    r = 50
    wu = np.float32(1.5) * np.float32(x[r + 1] - x[r])
    wd = np.float32(1.5) * np.float32(x[r] - x[r - 1])
    p = orc.default_params()
    p.link_dev2_max = 1e9
    on_edge = _event({r - 1: [(-wd, 0.0)], r: [(0.0, 0.0)], r + 1: [(wu, 0.0)]})
    res = orc.run(on_edge, p)
    assert res.link_up_raw[1] == 2 and res.link_dn_raw[1] == 0
    outside = _event({r - 1: [(-wd, 0.0)], r: [(0.0, 0.0)], r + 1: [(np.nextafter(wu, np.float32(10)), 0.0)]})
    res = orc.run(outside, p)
    assert res.link_up_raw[1] == -1 and res.link_dn_raw[1] == -1     # both or neither (R7)
    # z edge
    on_edge_z = _event({r - 1: [(0.0, wd)], r: [(0.0, 0.0)], r + 1: [(0.0, -wu)]})
    res = orc.run(on_edge_z, p)
    assert res.link_up_raw[1] == 2 and res.link_dn_raw[1] == 0


def test_deviation_cut():
    """Dev_best <= link_dev2_max links, above does not: kink of slope difference 0.8 -> Dev = 0.64 = the default cut."""
    r = 50
    dxu = float(np.float32(ROWX[r + 1]) - np.float32(ROWX[r]))
    dxd = float(np.float32(ROWX[r]) - np.float32(ROWX[r - 1]))
    p = orc.default_params()
    ev = _event({r - 1: [(0.0, 0.0)], r: [(0.0, 0.0)], r + 1: [(0.5 * dxu, 0.0)]})      # Dev = 0.25
    res = orc.run(ev, p)
    assert res.link_up_raw[1] == 2
    ev = _event({r - 1: [(0.0, 0.0)], r: [(0.0, 0.0)], r + 1: [(0.9 * dxu, 0.0)]})      # Dev = 0.81 > 0.64
    res = orc.run(ev, p)
    assert res.link_up_raw[1] == -1 and res.link_dn_raw[1] == -1
    assert dxd > 0


def test_dead_rows_are_bridged_r2():
    """R2: up(r) = first live row among r+1, r+2.  Collinear points across a dead row still link."""
    x = ROWX.astype(np.float64)
    dead = np.zeros(R, np.uint8)
    dead[41] = 1
    pts = {q: [(np.float32(0.1 * (x[q] - x[40])), np.float32(5.0))] for q in (39, 40, 42, 43)}
    ev = _event(pts, row_dead=dead)
    res = orc.run(ev)
    assert list(res.link_up_raw) == [-1, 2, 3, -1]
    assert list(res.link_dn_raw) == [-1, 0, 1, -1]
    # two dead rows in sequence are not bridged
    dead[42] = 1
    pts = {q: [(np.float32(0.1 * (x[q] - x[40])), np.float32(5.0))] for q in (39, 40, 43, 44)}
    res = orc.run(_event(pts, row_dead=dead))
    assert np.all(res.link_up_raw == -1)


# ------------------------------------------------------------------------------------------------ O3
@pytest.mark.parametrize("idx,scale", [(1, 0.05), (2, 0.05), (3, 0.04)])
def test_cleaned_links_are_reciprocal_paths(idx, scale):
    """north_star check 5 + path invariants (SURVEY.md 8(c) pins row O3)."""
    ev = datagen.make_event(idx, scale=scale)
    res = orc.run(ev)
    up, dn = res.link_up, res.link_dn
    n = ev.n_clusters
    h = np.arange(n)
    has_up = up >= 0
    assert np.array_equal(dn[up[has_up]], h[has_up])
    has_dn = dn >= 0
    assert np.array_equal(up[dn[has_dn]], h[has_dn])
    # cleaned links are a subset of the raw ones
    assert np.all((up == res.link_up_raw) | (up == -1)) and np.all((dn == res.link_dn_raw) | (dn == -1))
    # idempotence: cleaning the cleaned arrays changes nothing
    up2 = np.where(has_up & (dn[np.where(has_up, up, 0)] == h), up, -1)
    assert np.array_equal(up2, up)
    # links go strictly up in row, inside the sector
    bucket = np.repeat(np.arange(ev.n_sectors * R), np.diff(ev.row_offset.astype(np.int64)))
    assert np.all(bucket[up[has_up]] == bucket[has_up] + 1)            # no dead rows here: exactly one row up
    assert np.all(bucket[up[has_up]] // R == bucket[has_up] // R)
    # vertex-disjoint simple paths: in-degree <= 1
    assert np.unique(up[has_up]).size == has_up.sum()
    # start hits: heads of paths with >= 2 nodes, ascending global index
    heads = h[(~has_dn) & has_up]
    assert np.array_equal(res.start_hits, heads)
    assert len(heads) > 0


def test_empty_and_degenerate_inputs():
    """R24: empty events / rows / sectors are valid and give nothing."""
    ev = datagen.event_from_arrays(np.zeros(R + 1, np.uint32), [], [], 1, R)
    res = orc.run(ev)
    assert res.n_tracks == 0 and res.start_hits.size == 0
    ev = _event({10: [(0.0, 0.0)]})
    res = orc.run(ev)
    assert res.n_tracks == 0 and res.link_up_raw[0] == -1
    # clusters only on the first and last rows: no up/down row pair exists
    ev = _event({0: [(0.0, 0.0)], R - 1: [(0.0, 0.0)]})
    assert np.all(orc.run(ev).link_up_raw == -1)


def test_non_finite_input_is_rejected():
    ev = _event({10: [(float("nan"), 0.0)]})
    with pytest.raises(ValueError):
        orc.run(ev)


def test_o2_operation_counters_on_a_hand_case():
    """The O2 counters behind bench.py's operation count of the neighbour finder (no arithmetic depends on them): three
    collinear clusters on rows 10, 11, 12 plus one far-away cluster on row 11.  Every cluster has a row above and below (4);
    up candidates: the cluster of row 10 sees 1 (the far one is outside its window), that of row 11 sees 1, the far one 0,
    row 12 none: 2; down candidates likewise 2; pairs: 1 * 0 + 1 * 1 + 0 * 0 + 0 * 1 = 1."""
    from paper_1910_12214_b200.datagen import default_row_x
    X = default_row_x()
    counts = np.zeros(152, np.int64)
    counts[10], counts[11], counts[12] = 1, 2, 1
    off = np.concatenate([[0], np.cumsum(counts)])
    y = [0.0, 0.3 * (X[11] - X[10]), 40.0, 0.3 * (X[12] - X[10])]
    z = [5.0, 5.0, -100.0, 5.0]
    res = orc.run(datagen.event_from_arrays(off, y, z, 1, 152))
    assert res.o2_ops.tolist() == [4, 2, 2, 1]
    assert res.link_up_raw.tolist() == [-1, 3, -1, -1] and res.link_dn_raw.tolist() == [-1, 0, -1, -1]
    assert res.link_up.tolist() == [-1] * 4            # the end clusters have no pair, so nothing is reciprocal
