"""GPU-vs-oracle comparison used by the -m gpu parity tests (BASELINE.json north_star bars).

Bit-exact: neighbour links (raw and cleaned), start hits, tracklet status / hit counts / row spans / per-row
cluster indices, track count, per-track cluster-index lists and bookkeeping.  Floating point: track and
tracklet parameters within 1e-4 relative, covariances within 1e-3 relative (north_star).  With DESIGN.md R0
honoured on both sides the parameters are in fact expected to be bit-identical; `exact` reports that.
"""
import numpy as np

PAR_RTOL = 1e-4
COV_RTOL = 1e-3


def rel_err(a, b, floor):
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    if a.size == 0:
        return 0.0
    return float(np.max(np.abs(a - b) / np.maximum(np.maximum(np.abs(a), np.abs(b)), floor)))


def compare(gpu: dict, orc, n_rows: int, check_stages: bool = True) -> dict:
    """gpu: TrackResult.numpy() (with stages if check_stages); orc: oracle.tpc_oracle.OracleResult."""
    rep = {}
    if check_stages:
        for k in ("link_up_raw", "link_dn_raw", "link_up", "link_dn"):
            assert np.array_equal(gpu[k], getattr(orc, k)), k
        assert np.array_equal(gpu["start_hits"].view(np.uint32), orc.start_hits), "start_hits"
        assert np.array_equal(gpu["tl_status"], orc.tl_status), "tl_status"
        assert np.array_equal(gpu["tl_nhits"], orc.tl_nhits), "tl_nhits"
        assert np.array_equal(gpu["tl_first_row"], orc.tl_first_row), "tl_first_row"
        assert np.array_equal(gpu["tl_last_row"], orc.tl_last_row), "tl_last_row"
        assert np.array_equal(gpu["tl_rowhit"], orc.tl_rowhit), "tl_rowhit"
        acc = orc.tl_status == 2
        rep["tl_par_rel"] = rel_err(gpu["tl_par"][acc], orc.tl_par[acc], 1e-3)
        rep["tl_cov_rel"] = rel_err(gpu["tl_cov"][acc], orc.tl_cov[acc], 1e-9)
        rep["tl_exact"] = bool(np.array_equal(gpu["tl_par"][acc], orc.tl_par[acc].astype(np.float32)) and
                               np.array_equal(gpu["tl_cov"][acc], orc.tl_cov[acc].astype(np.float32)) and
                               np.array_equal(gpu["tl_chi2"][acc], orc.tl_chi2[acc].astype(np.float32)))
    # tracks
    assert gpu["trk_ncl"].shape[0] == orc.n_tracks, ("track count", gpu["trk_ncl"].shape[0], orc.n_tracks)
    assert np.array_equal(gpu["trk_tracklet"], orc.trk_tracklet), "trk_tracklet"
    assert np.array_equal(gpu["trk_sector"], orc.trk_sector), "trk_sector"
    assert np.array_equal(gpu["trk_first_row"], orc.trk_first_row), "trk_first_row"
    assert np.array_equal(gpu["trk_last_row"], orc.trk_last_row), "trk_last_row"
    assert np.array_equal(gpu["trk_ncl"], orc.trk_ncl), "trk_ncl"
    assert np.array_equal(gpu["trk_cl_offset"].view(np.uint32), orc.trk_cl_offset), "trk_cl_offset"
    assert np.array_equal(gpu["trk_cl_index"].view(np.uint32), orc.trk_cl_index), "trk_cl_index"
    par = gpu["trk_par"].T      # [n,5]
    cov = gpu["trk_cov"].T      # [n,15]
    rep["par_rel"] = rel_err(par, orc.trk_par, 1e-3)
    rep["cov_rel"] = rel_err(cov, orc.trk_cov, 1e-9)
    rep["x_exact"] = bool(np.array_equal(gpu["trk_x"], orc.trk_x.astype(np.float32)))
    rep["chi2_rel"] = rel_err(gpu["trk_chi2"], orc.trk_chi2, 1e-6)
    rep["exact"] = bool(np.array_equal(par, orc.trk_par.astype(np.float32)) and
                        np.array_equal(cov, orc.trk_cov.astype(np.float32)) and
                        np.array_equal(gpu["trk_chi2"], orc.trk_chi2.astype(np.float32)))
    assert rep["par_rel"] <= PAR_RTOL, rep
    assert rep["cov_rel"] <= COV_RTOL, rep
    assert rep["chi2_rel"] <= PAR_RTOL, rep
    assert rep["x_exact"], rep
    if check_stages:
        assert rep["tl_par_rel"] <= PAR_RTOL and rep["tl_cov_rel"] <= COV_RTOL, rep
    return rep
