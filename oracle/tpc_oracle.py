"""ctypes wrapper of the CPU oracle (oracle/tpc_oracle.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It does not import the CUDA package (only plain numpy arrays come in).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpc_oracle.cpp")
_HDR = os.path.join(_HERE, "tpc_oracle.h")
_LIB = os.path.join(_HERE, "libtpcoracle.so")

BRUTE_FORCE = 1
FP64 = 2
REFIT = 4
MERGE = 8
FLAGS = 16
LEGS = 32
MERGED = 64


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off -fno-fast-math (R0: no FMA contraction, no reassociation)."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", _SRC, "-o", _LIB])
    return _LIB


class Geometry(ctypes.Structure):
    _fields_ = [("n_sectors", ctypes.c_int32), ("n_rows", ctypes.c_int32), ("row_x", ctypes.c_void_p),
                ("row_dead", ctypes.c_void_p), ("bz_tesla", ctypes.c_float), ("tan_half_sector", ctypes.c_float),
                ("z_min", ctypes.c_float), ("z_max", ctypes.c_float)]


class Params(ctypes.Structure):
    _fields_ = [(n, ctypes.c_float) for n in
                ("area_y", "area_z", "link_dev2_max", "err2_y", "err2_z", "init_var_s", "init_var_t", "init_var_q",
                 "turn_var_scale", "max_sinphi", "road_sigma", "road_min", "road_max")] + \
               [(n, ctypes.c_int32) for n in ("max_row_gap", "min_chain_hits", "min_tracklet_hits", "min_track_hits")] + \
               [("cell_min", ctypes.c_float), ("cell_max", ctypes.c_float), ("merge_max_row_gap", ctypes.c_int32),
                ("merge_back_rows", ctypes.c_int32), ("merge_chi2_max", ctypes.c_float), ("tube_radius", ctypes.c_float),
                ("inv_pt_protect", ctypes.c_float),
                ("leg_min_sinphi", ctypes.c_float), ("leg_chi2_max", ctypes.c_float), ("leg_max_sectors", ctypes.c_int32),
                ("leg_max_row_diff", ctypes.c_int32), ("leg_max_centre_dist", ctypes.c_float), ("tube_chi2_max", ctypes.c_float)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        # TPC_ORACLE_LIB: another build of the same source (tests/test_oracle_sanitized.py loads one made with
        # -fsanitize=address,undefined); the arithmetic flags of that build are the test's business
        override = os.environ.get("TPC_ORACLE_LIB")
        if not override:
            build()
        L = ctypes.CDLL(override or _LIB)
        vp, i64, dbl, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int
        L.orcDefaultParams.argtypes = [ctypes.POINTER(Params)]
        L.orcDefaultParams.restype = None
        L.orcRun.argtypes = [ctypes.POINTER(Geometry), ctypes.POINTER(Params), i64, vp, vp, vp, ci, ctypes.POINTER(vp)]
        L.orcRun.restype = ci
        L.orcFree.argtypes = [vp]
        L.orcFree.restype = None
        for f in ("orcNumClusters", "orcNumStartHits", "orcNumTracks", "orcNumTrackClusters"):
            getattr(L, f).argtypes = [vp]
            getattr(L, f).restype = i64
        L.orcGetGrid.argtypes = [vp] * 4
        L.orcGetLinks.argtypes = [vp] * 5
        L.orcGetO4Counts.argtypes = [vp] * 2
        L.orcGetO4Counts.restype = None
        L.orcGetO2Counts.argtypes = [vp] * 2
        L.orcGetO2Counts.restype = None
        L.orcGetStartHits.argtypes = [vp] * 2
        L.orcGetTracklets.argtypes = [vp] * 10
        L.orcGetTracks.argtypes = [vp] * 12
        for f in ("orcGetGrid", "orcGetLinks", "orcGetStartHits", "orcGetTracklets", "orcGetTracks"):
            getattr(L, f).restype = None
        L.orcPackCharge.argtypes = [i64, vp, ci, vp]
        L.orcPackCharge.restype = ci
        L.orcPackPositions.argtypes = [i64, vp, vp, ci, vp]
        L.orcPackPositions.restype = ci
        L.orcGetResiduals.argtypes = [vp] * 3
        L.orcGetResiduals.restype = None
        L.orcGetClusterFlags.argtypes = [vp] * 3
        L.orcGetClusterFlags.restype = None
        L.orcGetMerge.argtypes = [vp] * 5
        L.orcGetMerge.restype = None
        L.orcRotate.argtypes = [vp, vp, dbl, dbl, dbl, ci]
        L.orcRotate.restype = ci
        L.orcMatch.argtypes = [ctypes.POINTER(Params), dbl, vp, vp, ci, vp, vp, ci, vp]
        L.orcMatch.restype = ci
        L.orcGetLegs.argtypes = [vp] * 3
        L.orcGetLegs.restype = None
        L.orcGetMerged.argtypes = [vp] * 5
        L.orcGetMerged.restype = None
        L.orcMirror.argtypes = [vp, vp]
        L.orcMirror.restype = None
        L.orcLegMatch.argtypes = [ctypes.POINTER(Params), dbl, vp, vp, ci, vp, vp, ci, vp]
        L.orcLegMatch.restype = ci
        L.orcGetRefit.argtypes = [vp] * 9
        L.orcGetRefit.restype = None
        L.orcRefitPoints.argtypes = [ctypes.POINTER(Geometry), ctypes.POINTER(Params), ci, vp, vp, vp, ci, vp, vp]
        L.orcRefitPoints.restype = ci
        L.orcSearch.argtypes = [ctypes.POINTER(Geometry), ctypes.POINTER(Params), ci, vp, vp, vp, ci, vp, vp, ci, ci]
        L.orcSearch.restype = ci
        L.orcPropagate.argtypes = [vp, vp, dbl, dbl, dbl, ci]
        L.orcPropagate.restype = ci
        L.orcUpdate.argtypes = [vp, vp, vp, dbl, dbl, dbl, dbl, ci]
        L.orcUpdate.restype = ci
        _lib = L
    return _lib


def default_params() -> Params:
    p = Params()
    _load().orcDefaultParams(ctypes.byref(p))
    return p


@dataclass
class OracleResult:
    n_clusters: int
    sorted_to_orig: np.ndarray
    cell_of_sorted: np.ndarray
    n_cells: np.ndarray
    link_up_raw: np.ndarray
    link_dn_raw: np.ndarray
    link_up: np.ndarray
    link_dn: np.ndarray
    start_hits: np.ndarray
    tl_status: np.ndarray
    tl_nhits: np.ndarray
    tl_first_row: np.ndarray
    tl_last_row: np.ndarray
    tl_rowhit: np.ndarray      # [n_start, n_rows]
    tl_x: np.ndarray
    tl_par: np.ndarray         # [n_start, 5]
    tl_cov: np.ndarray         # [n_start, 15]
    tl_chi2: np.ndarray
    trk_tracklet: np.ndarray
    trk_sector: np.ndarray
    trk_first_row: np.ndarray
    trk_last_row: np.ndarray
    trk_ncl: np.ndarray
    trk_x: np.ndarray
    trk_par: np.ndarray        # [n_tracks, 5]
    trk_cov: np.ndarray        # [n_tracks, 15]
    trk_chi2: np.ndarray
    trk_cl_offset: np.ndarray
    trk_cl_index: np.ndarray
    # O6 refit (only with refit=True): status, inner state (down pass), outer state (up pass)
    rf_status: np.ndarray | None = None
    rf_x_in: np.ndarray | None = None
    rf_par_in: np.ndarray | None = None     # [n_tracks, 5]
    rf_cov_in: np.ndarray | None = None     # [n_tracks, 15]
    rf_chi2: np.ndarray | None = None
    rf_x_out: np.ndarray | None = None
    rf_par_out: np.ndarray | None = None
    rf_cov_out: np.ndarray | None = None
    # O7 merger (only with merge=True): links between track segments
    mg_next: np.ndarray | None = None
    mg_prev: np.ndarray | None = None
    mg_head: np.ndarray | None = None
    mg_chi2: np.ndarray | None = None
    # O10 looper legs (only with legs=True): the track on the other side of the outer turn, chi2 of the pair
    lg_partner: np.ndarray | None = None
    lg_chi2: np.ndarray | None = None
    # O12 merged tracks (only with merged=True): merged-track id and leg rank per track, cluster lists along the path
    mt_id: np.ndarray | None = None
    mt_rank: np.ndarray | None = None
    mt_cl_offset: np.ndarray | None = None
    mt_cl_index: np.ndarray | None = None
    # O8 cluster flags (only with flags=True): bit mask per cluster and the owning track
    cf_flags: np.ndarray | None = None
    cf_owner: np.ndarray | None = None
    cf_res_y: np.ndarray | None = None      # track-model residuals of the clusters attached to refitted tracks
    cf_res_z: np.ndarray | None = None
    cf_res_code: np.ndarray | None = None   # O11: the residuals as 16-bit integers (y16 | z16 << 16), pos_bits of the call
    o4_ops: np.ndarray | None = None        # O4: Propagates, Updates, Searches, clusters inside the roads (counters only)
    o2_ops: np.ndarray | None = None        # O2: clusters with a row pair, up candidates, down candidates, pairs (counters only)

    @property
    def n_tracks(self) -> int:
        return int(self.trk_ncl.shape[0])


def _ptr(a):
    return a.ctypes.data if a is not None and a.size else None


def run(ev, params: Params | None = None, brute_force: bool = False, fp64: bool = False,
        stages_only: bool = False, refit: bool = False, merge: bool = False, flags: bool = False,
        legs: bool = False, pos_bits: int = 6, merged: bool = False) -> OracleResult:
    """Run O1..O5 on an Event-like object (fields n_sectors, n_rows, row_x, row_dead, bz_tesla,
    tan_half_sector, z_min, z_max, row_offset, y, z; numpy arrays)."""
    L = _load()
    p = params if params is not None else default_params()
    row_x = np.ascontiguousarray(ev.row_x, np.float32)
    dead = np.ascontiguousarray(ev.row_dead, np.uint8)
    g = Geometry(ev.n_sectors, ev.n_rows, row_x.ctypes.data, dead.ctypes.data if dead.any() else None, ev.bz_tesla,
                 ev.tan_half_sector, ev.z_min, ev.z_max)
    off = np.ascontiguousarray(ev.row_offset, np.uint32)
    y = np.ascontiguousarray(ev.y, np.float32)
    z = np.ascontiguousarray(ev.z, np.float32)
    n = int(y.shape[0])
    h = ctypes.c_void_p()
    rc = L.orcRun(ctypes.byref(g), ctypes.byref(p), n, off.ctypes.data, _ptr(y), _ptr(z),
                  (BRUTE_FORCE if brute_force else 0) | (FP64 if fp64 else 0) | (REFIT if refit else 0) | (MERGE if merge else 0) | (FLAGS if flags else 0) | (LEGS if legs else 0) | (MERGED if merged else 0),
                  ctypes.byref(h))
    if rc != 0:
        raise ValueError(f"orcRun failed with {rc}")
    try:
        R = ev.n_rows
        ns, nt, ntc = L.orcNumStartHits(h), L.orcNumTracks(h), L.orcNumTrackClusters(h)
        ng = 0 if brute_force else n
        s2o, cell = np.zeros(ng, np.uint32), np.zeros(ng, np.int32)
        ncell = np.zeros(ev.n_sectors * R if not brute_force else 0, np.int32)
        L.orcGetGrid(h, _ptr(s2o), _ptr(cell), _ptr(ncell))
        ur, dr, u, d = (np.full(n, -1, np.int32) for _ in range(4))
        L.orcGetLinks(h, _ptr(ur), _ptr(dr), _ptr(u), _ptr(d))
        sh = np.zeros(ns, np.uint32)
        L.orcGetStartHits(h, _ptr(sh))
        st, nh, fr, lr = (np.zeros(ns, np.int32) for _ in range(4))
        rh = np.full((ns, R), -1, np.int32)
        tx, tchi = np.zeros(ns), np.zeros(ns)
        tpar, tcov = np.zeros((ns, 5)), np.zeros((ns, 15))
        L.orcGetTracklets(h, _ptr(st), _ptr(nh), _ptr(fr), _ptr(lr), _ptr(rh), _ptr(tx), _ptr(tpar), _ptr(tcov),
                          _ptr(tchi))
        kid, ks, kf, kl, kn = (np.zeros(nt, np.int32) for _ in range(5))
        kx, kchi = np.zeros(nt), np.zeros(nt)
        kpar, kcov = np.zeros((nt, 5)), np.zeros((nt, 15))
        koff, kidx = np.zeros(nt + 1, np.uint32), np.zeros(ntc, np.uint32)
        L.orcGetTracks(h, _ptr(kid), _ptr(ks), _ptr(kf), _ptr(kl), _ptr(kn), _ptr(kx), _ptr(kpar), _ptr(kcov),
                       _ptr(kchi), _ptr(koff), _ptr(kidx))
        rf = {}
        ops = np.zeros(4, np.int64)
        L.orcGetO4Counts(h, _ptr(ops))
        rf["o4_ops"] = ops
        ops2 = np.zeros(4, np.int64)
        L.orcGetO2Counts(h, _ptr(ops2))
        rf["o2_ops"] = ops2
        merge = merge or merged
        legs = legs or merged
        refit = refit or merge or flags or legs
        if refit:
            rst = np.zeros(nt, np.int32)
            rxi, rchi, rxo = np.zeros(nt), np.zeros(nt), np.zeros(nt)
            rpi, rpo, rci, rco = np.zeros((nt, 5)), np.zeros((nt, 5)), np.zeros((nt, 15)), np.zeros((nt, 15))
            L.orcGetRefit(h, _ptr(rst), _ptr(rxi), _ptr(rpi), _ptr(rci), _ptr(rchi), _ptr(rxo), _ptr(rpo), _ptr(rco))
            rf.update(rf_status=rst, rf_x_in=rxi, rf_par_in=rpi, rf_cov_in=rci, rf_chi2=rchi, rf_x_out=rxo, rf_par_out=rpo,
                      rf_cov_out=rco)
        if merge:
            mn, mp, mh = (np.full(nt, -1, np.int32) for _ in range(3))
            mc = np.zeros(nt)
            L.orcGetMerge(h, _ptr(mn), _ptr(mp), _ptr(mh), _ptr(mc))
            rf.update(mg_next=mn, mg_prev=mp, mg_head=mh, mg_chi2=mc)
        if legs:
            lp, lc = np.full(nt, -1, np.int32), np.zeros(nt)
            L.orcGetLegs(h, _ptr(lp), _ptr(lc))
            rf.update(lg_partner=lp, lg_chi2=lc)
        if merged:
            mi, mr = np.full(nt, -1, np.int32), np.zeros(nt, np.int32)
            mo, mx = np.zeros(nt + 1, np.uint32), np.zeros(ntc, np.uint32)
            L.orcGetMerged(h, _ptr(mi), _ptr(mr), _ptr(mo), _ptr(mx))
            rf.update(mt_id=mi, mt_rank=mr, mt_cl_offset=mo, mt_cl_index=mx)
        if flags:
            cf, co = np.zeros(n, np.uint8), np.full(n, -1, np.int32)
            L.orcGetClusterFlags(h, _ptr(cf), _ptr(co))
            ry, rz = np.zeros(n), np.zeros(n)
            L.orcGetResiduals(h, _ptr(ry), _ptr(rz))
            rf.update(cf_flags=cf, cf_owner=co, cf_res_y=ry, cf_res_z=rz)
    finally:
        L.orcFree(h)
    if flags:        # O11: the residuals in the 16-bit integer format
        rf["cf_res_code"] = pack_positions(rf["cf_res_y"].astype(np.float32), rf["cf_res_z"].astype(np.float32), pos_bits)
    return OracleResult(n, s2o, cell, ncell, ur, dr, u, d, sh, st, nh, fr, lr, rh, tx, tpar, tcov, tchi, kid, ks, kf, kl,
                        kn, kx, kpar, kcov, kchi, koff, kidx, **rf)


def propagate(state, cov, x_new, bz_tesla=0.5, max_sinphi=0.98, fp64=True):
    """One Propagate step.  state = (x, y, z, s, t, q); cov = 15 lower-triangle elements.  Returns (ok, state, cov)."""
    s = np.array(state, np.float64)
    c = np.array(cov, np.float64)
    ok = _load().orcPropagate(s.ctypes.data, c.ctypes.data, float(x_new), float(bz_tesla), float(max_sinphi), int(fp64))
    return bool(ok), s, c


def update(state, cov, chi2, ym, zm, err2_y=0.01, err2_z=0.01, fp64=True):
    """One Update step (y then z).  Returns (ok, state, cov, chi2)."""
    s = np.array(state, np.float64)
    c = np.array(cov, np.float64)
    x2 = np.array([chi2], np.float64)
    ok = _load().orcUpdate(s.ctypes.data, c.ctypes.data, x2.ctypes.data, float(ym), float(zm), float(err2_y),
                           float(err2_z), int(fp64))
    return bool(ok), s, c, float(x2[0])


def search(rows, y, z, row, state, cov, row_x, params: Params | None = None, fp64=False, brute=False, bz_tesla=0.5):
    """One O4 Search among the given clusters of one sector (ascending rows).  Returns the picked index or -1."""
    p = params if params is not None else default_params()
    row_x = np.ascontiguousarray(row_x, np.float32)
    g = Geometry(1, len(row_x), row_x.ctypes.data, None, bz_tesla, float(np.tan(np.radians(10.0))), -250.0, 250.0)
    rows = np.ascontiguousarray(rows, np.int32)
    yy, zz = np.ascontiguousarray(y, np.float32), np.ascontiguousarray(z, np.float32)
    s, c = np.array(state, np.float64), np.array(cov, np.float64)
    rc = _load().orcSearch(ctypes.byref(g), ctypes.byref(p), len(rows), _ptr(rows), _ptr(yy), _ptr(zz), int(row),
                           s.ctypes.data, c.ctypes.data, int(fp64), int(brute))
    if rc == -2:
        raise ValueError("orcSearch: bad arguments")
    return int(rc)


def refit_points(rows, y, z, row_x, bz_tesla=0.5, params: Params | None = None, fp64=True):
    """O6 refit of the given clusters (ascending rows) of one sector.  Returns (ok, inner, outer), each state an
    array of 22 doubles: x, y, z, s, t, q, C[15], chi2."""
    L = _load()
    p = params if params is not None else default_params()
    row_x = np.ascontiguousarray(row_x, np.float32)
    g = Geometry(1, len(row_x), row_x.ctypes.data, None, bz_tesla, float(np.tan(np.radians(10.0))), -250.0, 250.0)
    rows = np.ascontiguousarray(rows, np.int32)
    yy, zz = np.ascontiguousarray(y, np.float64), np.ascontiguousarray(z, np.float64)
    inner, outer = np.zeros(22), np.zeros(22)
    ok = L.orcRefitPoints(ctypes.byref(g), ctypes.byref(p), len(rows), rows.ctypes.data, yy.ctypes.data, zz.ctypes.data,
                          int(fp64), inner.ctypes.data, outer.ctypes.data)
    return bool(ok), inner, outer


def rotate(state, cov, alpha, bz_tesla=0.5, max_sinphi=0.98, fp64=True):
    """O7 Rotate: the state seen from a frame turned by alpha (radians).  Returns (ok, state, cov)."""
    s = np.array(state, np.float64)
    c = np.array(cov, np.float64)
    ok = _load().orcRotate(s.ctypes.data, c.ctypes.data, float(alpha), float(bz_tesla), float(max_sinphi), int(fp64))
    return bool(ok), s, c


def match(a_state, a_cov, rel, b_state, b_cov, bz_tesla=0.5, params: Params | None = None, fp64=True):
    """O7 Match of outer state a to inner state b (rel = 0 same sector, +-1 neighbour).  Returns (ok, chi2)."""
    p = params if params is not None else default_params()
    a, ac = np.array(a_state, np.float64), np.array(a_cov, np.float64)
    b, bc = np.array(b_state, np.float64), np.array(b_cov, np.float64)
    chi2 = np.zeros(1)
    ok = _load().orcMatch(ctypes.byref(p), float(bz_tesla), a.ctypes.data, ac.ctypes.data, int(rel), b.ctypes.data,
                          bc.ctypes.data, int(fp64), chi2.ctypes.data)
    return bool(ok), float(chi2[0])


def mirror(state, cov):
    """O10 Mirror: the state seen from the frame turned by 180 degrees and walked backwards.  Returns (state, cov)."""
    s = np.array(state, np.float64)
    c = np.array(cov, np.float64)
    _load().orcMirror(s.ctypes.data, c.ctypes.data)
    return s, c


def leg_match(a_state, a_cov, d, b_state, b_cov, bz_tesla=0.5, params: Params | None = None, fp64=True):
    """O10 LegMatch of two outer states (b's sector d sectors after a's).  Returns (ok, chi2)."""
    p = params if params is not None else default_params()
    a, ac = np.array(a_state, np.float64), np.array(a_cov, np.float64)
    b, bc = np.array(b_state, np.float64), np.array(b_cov, np.float64)
    chi2 = np.zeros(1)
    ok = _load().orcLegMatch(ctypes.byref(p), float(bz_tesla), a.ctypes.data, ac.ctypes.data, int(d), b.ctypes.data,
                             bc.ctypes.data, int(fp64), chi2.ctypes.data)
    return bool(ok), float(chi2[0])


def pack_positions(y, z, bits=6):
    """O11: positions (or residuals) as 16-bit integers in units of 2^-bits cm; returns uint32 = y16 | z16 << 16."""
    y = np.ascontiguousarray(y, np.float32)
    z = np.ascontiguousarray(z, np.float32)
    code = np.zeros(y.shape[0], np.uint32)
    if y.shape != z.shape or not _load().orcPackPositions(y.shape[0], _ptr(y), _ptr(z), int(bits), _ptr(code)):
        raise ValueError("orcPackPositions: bad arguments")
    return code


def pack_charge(q, trunc_bits=4):
    """O9: dynamic-precision 16-bit code of the charges."""
    q = np.ascontiguousarray(q, np.float32)
    code = np.zeros(q.shape[0], np.uint16)
    if not _load().orcPackCharge(q.shape[0], _ptr(q), int(trunc_bits), _ptr(code)):
        raise ValueError("orcPackCharge: bad arguments")
    return code
