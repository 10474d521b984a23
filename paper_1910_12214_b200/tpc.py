"""Thin binding of libtpcgpu.so (include/tpc_abi.h): same names, argument marshalling only.

PyTorch is used for device memory and the stream, nothing else: every step of the path (grid, neighbour
finder, cleaner, tracklet constructor, selector) runs in the library's CUDA kernels.  There is no CPU
fallback: loading fails loudly when the library cannot be built or loaded.
"""
from __future__ import annotations

import ctypes
from ctypes import POINTER, byref, c_char_p, c_float, c_int, c_int32, c_int64, c_size_t, c_void_p
from dataclasses import dataclass

import numpy as np

from . import build as _build

TPC_OK = 0
TPC_ERR_INVALID_ARG = -1
TPC_ERR_UNSORTED_OFFSETS = -2
TPC_ERR_WORKSPACE_TOO_SMALL = -3
TPC_ERR_CAPACITY = -4
TPC_ERR_CUDA = -5
TPC_ERR_NONFINITE_INPUT = -6
TPC_ERR_OUT_OF_MEMORY = -7
TPC_ERR_NOALLOC_LIMIT = -8


class tpcGeometry(ctypes.Structure):
    _fields_ = [("n_sectors", c_int32), ("n_rows", c_int32), ("row_x", c_void_p), ("row_pitch", c_void_p),
                ("row_dead", c_void_p), ("bz_tesla", c_float), ("tan_half_sector", c_float), ("z_min", c_float),
                ("z_max", c_float)]


class tpcParams(ctypes.Structure):
    _fields_ = [(n, c_float) for n in ("area_y", "area_z", "link_dev2_max", "err2_y", "err2_z", "init_var_s",
                                       "init_var_t", "init_var_q", "turn_var_scale", "max_sinphi", "road_sigma",
                                       "road_min", "road_max")] + \
               [(n, c_int32) for n in ("max_row_gap", "min_chain_hits", "min_tracklet_hits", "min_track_hits")] + \
               [("cell_min", c_float), ("cell_max", c_float), ("clusters_per_cell", c_float),
                ("validate_input", c_int32), ("force_wide_keys", c_int32), ("merge_max_row_gap", c_int32),
                ("merge_back_rows", c_int32), ("merge_chi2_max", c_float), ("tube_radius", c_float),
                ("inv_pt_protect", c_float), ("charge_trunc_bits", c_int32), ("leg_min_sinphi", c_float),
                ("leg_chi2_max", c_float), ("leg_max_sectors", c_int32), ("leg_max_row_diff", c_int32),
                ("leg_max_centre_dist", c_float), ("pos_bits", c_int32), ("tube_chi2_max", c_float)]


class tpcClusters(ctypes.Structure):
    _fields_ = [("n_clusters", c_int64), ("row_offset", c_void_p), ("x", c_void_p), ("y", c_void_p), ("z", c_void_p),
                ("q", c_void_p)]


_TRK_PTRS = ("trk_tracklet", "trk_sector", "trk_first_row", "trk_last_row", "trk_ncl", "trk_x", "trk_par", "trk_cov",
             "trk_chi2", "trk_cl_offset", "trk_cl_index")
_STAGE_PTRS = ("link_up_raw", "link_dn_raw", "link_up", "link_dn", "start_hits", "tl_status", "tl_nhits",
               "tl_first_row", "tl_last_row", "tl_rowhit", "tl_x", "tl_par", "tl_cov", "tl_chi2")
_REFIT_PTRS = ("trk_rf_status", "trk_rf_x_in", "trk_rf_par_in", "trk_rf_cov_in", "trk_rf_chi2", "trk_rf_x_out",
               "trk_rf_par_out", "trk_rf_cov_out")
_MERGE_PTRS = ("trk_mg_next", "trk_mg_prev", "trk_mg_head", "trk_mg_chi2")
_LEG_PTRS = ("trk_leg_partner", "trk_leg_chi2")
_FLAG_PTRS = ("cl_flags", "cl_owner", "cl_res_y", "cl_res_z")
_PACK_PTRS = ("cl_qcode",)
_POS_PTRS = ("cl_pos_code", "cl_res_code")
_MERGED_PTRS = ("trk_mt_id", "trk_mt_rank", "mt_cl_offset", "mt_cl_index")


class tpcTracks(ctypes.Structure):
    _fields_ = [("cap_tracks", c_int64), ("cap_track_clusters", c_int64)] + \
               [(n, c_void_p) for n in _TRK_PTRS + _STAGE_PTRS + _REFIT_PTRS + _MERGE_PTRS + _LEG_PTRS + _FLAG_PTRS + _PACK_PTRS + _POS_PTRS + _MERGED_PTRS]


class tpcRunStatus(ctypes.Structure):
    _fields_ = [("status", c_int32), ("kernel_launches", c_int32), ("n_clusters", c_int64), ("n_start_hits", c_int64),
                ("n_tracklets", c_int64), ("n_tracklet_hits", c_int64), ("n_tracks", c_int64),
                ("n_track_clusters", c_int64), ("n_cells", c_int64), ("stage_ms", c_float * 8), ("merge_ms", c_float), ("pack_ms", c_float), ("flags_ms", c_float), ("legs_ms", c_float), ("merged_ms", c_float),
                ("submit_ms", c_float * 2)]


ABI_SYMBOLS = ("tpcDefaultParams", "tpcCreate", "tpcDestroy", "tpcWorkspaceBytes", "tpcRun", "tpcGetRunStatus",
               "tpcSetProfiling", "tpcRunHost", "tpcSubmitHost", "tpcCollectHost", "tpcErrorString", "tpcLastCudaError",
               "tpcSelfTestDivision", "tpcNoAllocMaxClusters", "tpcNoAllocSetup", "tpcStartHitsNoAlloc", "tpcNoAllocLastError")

_lib = None


def load_library(build_if_stale: bool = True) -> ctypes.CDLL:
    """dlopen libtpcgpu.so (building it with nvcc when missing or older than its sources)."""
    global _lib
    if _lib is not None:
        return _lib
    import os
    path = os.environ.get("TPCGPU_LIB")          # tuning variants (build.build_cuda(out=...)); default: the product
    if not path:
        path = _build.LIB
        if build_if_stale:
            _build.build_cuda()
    try:
        L = ctypes.CDLL(path)
    except OSError as e:   # no fallback: the product path needs the CUDA library
        raise RuntimeError(f"libtpcgpu.so could not be loaded ({e}); the TPC tracker has no CPU fallback") from e
    vp = c_void_p
    L.tpcDefaultParams.argtypes = [POINTER(tpcParams)]
    L.tpcCreate.argtypes = [POINTER(vp), POINTER(tpcGeometry), POINTER(tpcParams), c_int]
    L.tpcDestroy.argtypes = [vp]
    L.tpcWorkspaceBytes.argtypes = [vp, c_int64, c_int64, POINTER(c_size_t)]
    L.tpcRun.argtypes = [vp, POINTER(tpcClusters), POINTER(tpcTracks), c_int64, vp, c_size_t, vp]
    L.tpcGetRunStatus.argtypes = [vp, POINTER(tpcRunStatus)]
    L.tpcSetProfiling.argtypes = [vp, c_int]
    L.tpcRunHost.argtypes = [vp, c_int64, vp, vp, vp, POINTER(tpcTracks), POINTER(tpcRunStatus), vp]
    L.tpcSubmitHost.argtypes = [vp, c_int, c_int64, vp, vp, vp, POINTER(tpcTracks)]
    L.tpcCollectHost.argtypes = [vp, c_int, POINTER(tpcRunStatus)]
    for f in ABI_SYMBOLS[:10]:
        getattr(L, f).restype = c_int
    L.tpcErrorString.argtypes = [c_int]
    L.tpcErrorString.restype = c_char_p
    L.tpcLastCudaError.argtypes = [vp]
    L.tpcLastCudaError.restype = c_char_p
    L.tpcSelfTestDivision.argtypes = [vp, c_int64, ctypes.c_uint64, POINTER(c_int64), POINTER(c_int64)]
    L.tpcSelfTestDivision.restype = c_int
    L.tpcNoAllocMaxClusters.argtypes = []
    L.tpcNoAllocMaxClusters.restype = c_int64
    L.tpcNoAllocSetup.argtypes = [c_int]
    L.tpcNoAllocSetup.restype = c_int
    L.tpcStartHitsNoAlloc.argtypes = [c_int, c_int64, vp, vp, vp, c_int64, vp, vp]
    L.tpcStartHitsNoAlloc.restype = c_int
    L.tpcNoAllocLastError.argtypes = []
    L.tpcNoAllocLastError.restype = c_char_p
    _lib = L
    return L


class TpcError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        msg = load_library().tpcErrorString(code).decode()
        super().__init__(f"{where}: {msg} ({code})" + (f": {detail}" if detail else ""))


# ---- the ABI calls under their own names -------------------------------------------------------------------
def tpcDefaultParams() -> tpcParams:
    p = tpcParams()
    rc = load_library().tpcDefaultParams(byref(p))
    if rc != TPC_OK:
        raise TpcError(rc, "tpcDefaultParams")
    return p


def tpcCreate(geometry: tpcGeometry, params: tpcParams, cuda_device: int = 0) -> c_void_p:
    h = c_void_p()
    rc = load_library().tpcCreate(byref(h), byref(geometry), byref(params), cuda_device)
    if rc != TPC_OK:
        raise TpcError(rc, "tpcCreate")
    return h


def tpcDestroy(handle) -> None:
    load_library().tpcDestroy(handle)


def tpcWorkspaceBytes(handle, n_clusters: int, cap_tracklets: int) -> int:
    b = c_size_t()
    rc = load_library().tpcWorkspaceBytes(handle, n_clusters, cap_tracklets, byref(b))
    if rc != TPC_OK:
        raise TpcError(rc, "tpcWorkspaceBytes")
    return b.value


def tpcRun(handle, clusters: tpcClusters, tracks: tpcTracks, cap_tracklets: int, workspace_ptr: int,
           workspace_bytes: int, cuda_stream: int = 0) -> None:
    L = load_library()
    rc = L.tpcRun(handle, byref(clusters), byref(tracks), cap_tracklets, workspace_ptr, workspace_bytes, cuda_stream)
    if rc != TPC_OK:
        raise TpcError(rc, "tpcRun", L.tpcLastCudaError(handle).decode())


def tpcGetRunStatus(handle) -> tpcRunStatus:
    L = load_library()
    s = tpcRunStatus()
    rc = L.tpcGetRunStatus(handle, byref(s))
    if rc != TPC_OK:
        raise TpcError(rc, "tpcGetRunStatus", L.tpcLastCudaError(handle).decode())
    return s


def tpcSetProfiling(handle, on: bool) -> None:
    load_library().tpcSetProfiling(handle, int(on))


def tpcSelfTestDivision(handle, n_threads: int, seed: int = 1):
    """(operand pairs tested, bit patterns that differ between the shared-reciprocal division and the IEEE one)."""
    L = load_library()
    nt, nm = c_int64(), c_int64()
    rc = L.tpcSelfTestDivision(handle, int(n_threads), int(seed), byref(nt), byref(nm))
    if rc != TPC_OK:
        raise TpcError(rc, "tpcSelfTestDivision", L.tpcLastCudaError(handle).decode())
    return nt.value, nm.value


# ---- convenience wrapper: allocation of device tensors with torch, nothing else ---------------------------
def tpcNoAllocMaxClusters() -> int:
    return int(load_library().tpcNoAllocMaxClusters())


def tpcNoAllocSetup(cuda_device: int = 0) -> None:
    L = load_library()
    rc = L.tpcNoAllocSetup(cuda_device)
    if rc != TPC_OK:
        raise TpcError(rc, "tpcNoAllocSetup", L.tpcNoAllocLastError().decode())


def tpcStartHitsNoAlloc(cuda_device: int, n_clusters: int, link_up_ptr: int, link_dn_ptr: int, start_hits_ptr: int,
                        cap_start_hits: int, n_start_hits_ptr: int, cuda_stream: int = 0) -> None:
    """The allocation-free start-hit list (include/tpc_abi.h): DEVICE pointers as integers; enqueues and returns."""
    L = load_library()
    rc = L.tpcStartHitsNoAlloc(cuda_device, n_clusters, link_up_ptr or None, link_dn_ptr or None, start_hits_ptr or None,
                               cap_start_hits, n_start_hits_ptr or None, cuda_stream or None)
    if rc != TPC_OK:
        raise TpcError(rc, "tpcStartHitsNoAlloc", L.tpcNoAllocLastError().decode())


@dataclass
class TrackResult:
    """Device tensors (torch) of one tpcRun, trimmed to the counts of the run status."""
    status: tpcRunStatus
    n_tracks: int
    n_track_clusters: int
    trk: dict          # name -> torch tensor (device); trk_par [5,n], trk_cov [15,n]
    stages: dict       # optional per-stage outputs (device tensors), empty unless requested

    def numpy(self) -> dict:
        out = {k: v.cpu().numpy() for k, v in self.trk.items()}
        out.update({k: v.cpu().numpy() for k, v in self.stages.items()})
        return out


class TpcTracker:
    """Owns a tpcHandle plus torch-allocated workspace and output buffers (grown on demand)."""

    def __init__(self, n_sectors, n_rows, row_x, row_dead=None, row_pitch=None, bz_tesla=0.5,
                 tan_half_sector=0.17632698070846498, z_min=-250.0, z_max=250.0, params: tpcParams | None = None,
                 device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("TpcTracker needs a CUDA device (there is no CPU fallback)")
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.n_sectors, self.n_rows = int(n_sectors), int(n_rows)
        self._row_x = np.ascontiguousarray(row_x, np.float32)
        self._row_dead = None if row_dead is None else np.ascontiguousarray(row_dead, np.uint8)
        self._row_pitch = None if row_pitch is None else np.ascontiguousarray(row_pitch, np.float32)
        self.params = params if params is not None else tpcDefaultParams()
        g = tpcGeometry(self.n_sectors, self.n_rows, self._row_x.ctypes.data,
                        None if self._row_pitch is None else self._row_pitch.ctypes.data,
                        None if self._row_dead is None else self._row_dead.ctypes.data, bz_tesla, tan_half_sector,
                        z_min, z_max)
        self.handle = tpcCreate(g, self.params, device)
        self._ws = None
        self._out = {}
        self._caps = (0, 0, 0)

    @classmethod
    def from_event(cls, ev, params: tpcParams | None = None, device: int = 0) -> "TpcTracker":
        return cls(ev.n_sectors, ev.n_rows, ev.row_x, ev.row_dead if np.any(ev.row_dead) else None, ev.row_pitch,
                   ev.bz_tesla, ev.tan_half_sector, ev.z_min, ev.z_max, params, device)

    def close(self):
        if getattr(self, "handle", None):
            tpcDestroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_profiling(self, on: bool):
        tpcSetProfiling(self.handle, on)

    def upload(self, ev):
        """Copy an Event's row_offset / y / z to the device (torch tensors; int32 view of the uint32 offsets)."""
        t = self.torch
        off = t.from_numpy(np.ascontiguousarray(ev.row_offset, np.uint32).view(np.int32)).to(self.device)
        y = t.from_numpy(np.ascontiguousarray(ev.y, np.float32)).to(self.device)
        z = t.from_numpy(np.ascontiguousarray(ev.z, np.float32)).to(self.device)
        return off, y, z

    def _ensure(self, n, capT, capK, capC, stages, refit=False, merge=False, flags=False, pack=False, legs=False, pos=False,
                merged=False):
        t = self.torch
        need = tpcWorkspaceBytes(self.handle, n, capT)
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = t.empty(need, dtype=t.uint8, device=self.device)
        i32, f32 = t.int32, t.float32
        spec = {"trk_tracklet": ((capK,), i32), "trk_sector": ((capK,), i32), "trk_first_row": ((capK,), i32),
                "trk_last_row": ((capK,), i32), "trk_ncl": ((capK,), i32), "trk_x": ((capK,), f32),
                "trk_par": ((5, capK), f32), "trk_cov": ((15, capK), f32), "trk_chi2": ((capK,), f32),
                "trk_cl_offset": ((capK + 1,), i32), "trk_cl_index": ((max(capC, 1),), i32)}
        if stages:
            R = self.n_rows
            spec.update({"link_up_raw": ((max(n, 1),), i32), "link_dn_raw": ((max(n, 1),), i32),
                         "link_up": ((max(n, 1),), i32), "link_dn": ((max(n, 1),), i32),
                         "start_hits": ((capT,), i32), "tl_status": ((capT,), i32), "tl_nhits": ((capT,), i32),
                         "tl_first_row": ((capT,), i32), "tl_last_row": ((capT,), i32), "tl_rowhit": ((capT, R), i32),
                         "tl_x": ((capT,), f32), "tl_par": ((capT, 5), f32), "tl_cov": ((capT, 15), f32),
                         "tl_chi2": ((capT,), f32)})
        if refit:
            spec.update({"trk_rf_status": ((capK,), i32), "trk_rf_x_in": ((capK,), f32), "trk_rf_par_in": ((5, capK), f32),
                         "trk_rf_cov_in": ((15, capK), f32), "trk_rf_chi2": ((capK,), f32), "trk_rf_x_out": ((capK,), f32),
                         "trk_rf_par_out": ((5, capK), f32), "trk_rf_cov_out": ((15, capK), f32)})
        if pack:
            spec.update({"cl_qcode": ((max(n, 1),), t.int16)})
        if flags:
            spec.update({"cl_flags": ((max(n, 1),), t.uint8), "cl_owner": ((max(n, 1),), i32),
                         "cl_res_y": ((max(n, 1),), f32), "cl_res_z": ((max(n, 1),), f32)})
        if merge:
            spec.update({"trk_mg_next": ((capK,), i32), "trk_mg_prev": ((capK,), i32), "trk_mg_head": ((capK,), i32),
                         "trk_mg_chi2": ((capK,), f32)})
        if pos:
            spec.update({"cl_pos_code": ((max(n, 1),), i32)})
            if flags:
                spec.update({"cl_res_code": ((max(n, 1),), i32)})
        if legs:
            spec.update({"trk_leg_partner": ((capK,), i32), "trk_leg_chi2": ((capK,), f32)})
        if merged:
            spec.update({"trk_mt_id": ((capK,), i32), "trk_mt_rank": ((capK,), i32), "mt_cl_offset": ((capK + 1,), i32),
                         "mt_cl_index": ((max(capC, 1),), i32)})
        for k, (shape, dt) in spec.items():
            cur = self._out.get(k)
            if cur is None or tuple(cur.shape) != shape:
                self._out[k] = t.empty(shape, dtype=dt, device=self.device)
        for k in list(self._out):
            if k not in spec:
                del self._out[k]

    def run(self, row_offset, y, z, cap_tracklets: int | None = None, cap_tracks: int | None = None,
            cap_track_clusters: int | None = None, stages: bool = False, stream=None, sync: bool = True,
            grow: bool = True, refit: bool = False, merge: bool = False, flags: bool = False, q=None,
            legs: bool = False, pos: bool = False, merged: bool = False):
        """One tpcRun on device tensors (q: optional device tensor of charges -> cl_qcode, the O9 charge code).  Returns a TrackResult (after synchronising) or None when sync=False."""
        t = self.torch
        n = int(y.shape[0])
        merge = merge or merged                   # the merged tracks are built from the merger's chains and the leg pairs
        legs = legs or merged
        refit = refit or merge or flags or legs   # the merger, the leg pairs and the cluster flags work on the refitted states
        capT = int(cap_tracklets) if cap_tracklets is not None else max(4096, n // 8)
        capK = int(cap_tracks) if cap_tracks is not None else capT
        capC = int(cap_track_clusters) if cap_track_clusters is not None else max(n, 1)
        attempts = 3 if grow else 0     # a too-small cap_tracklets hides the true track counts: up to 3 rounds
        while True:
            self._ensure(n, capT, capK, capC, stages, refit, merge, flags, q is not None, legs, pos, merged)
            cl = tpcClusters(n, row_offset.data_ptr(), None, y.data_ptr() if n else None, z.data_ptr() if n else None,
                             q.data_ptr() if (q is not None and n) else None)
            tr = tpcTracks()
            tr.cap_tracks, tr.cap_track_clusters = capK, capC
            for k, v in self._out.items():
                setattr(tr, k, v.data_ptr())
            s = stream if stream is not None else t.cuda.current_stream(self.device)
            tpcRun(self.handle, cl, tr, capT, self._ws.data_ptr(), self._ws.numel(), s.cuda_stream)
            if not sync:
                return None
            st = tpcGetRunStatus(self.handle)
            if st.status == TPC_ERR_CAPACITY and attempts > 0:
                capT = max(capT, st.n_start_hits)
                capK = max(capK, st.n_tracks)
                capC = max(capC, st.n_track_clusters)
                attempts -= 1
                continue
            break
        if st.status not in (TPC_OK, TPC_ERR_CAPACITY):
            raise TpcError(st.status, "tpcRun (device status)")
        nt = min(int(st.n_tracks), capK)
        nc = min(int(st.n_track_clusters), capC)
        ns = min(int(st.n_start_hits), capT)
        o = self._out
        trk = {k: (o[k][:, :nt] if o[k].dim() == 2 else o[k][:nt]) for k in _TRK_PTRS[:9]}
        trk["trk_cl_offset"] = o["trk_cl_offset"][:nt + 1]
        trk["trk_cl_index"] = o["trk_cl_index"][:nc]
        if refit:
            for k in _REFIT_PTRS:
                trk[k] = o[k][:, :nt] if o[k].dim() == 2 else o[k][:nt]
        if merge:
            for k in _MERGE_PTRS:
                trk[k] = o[k][:nt]
        if legs:
            for k in _LEG_PTRS:
                trk[k] = o[k][:nt]
        if merged:
            trk["trk_mt_id"], trk["trk_mt_rank"] = o["trk_mt_id"][:nt], o["trk_mt_rank"][:nt]
            trk["mt_cl_offset"], trk["mt_cl_index"] = o["mt_cl_offset"][:nt + 1], o["mt_cl_index"][:nc]
        if flags:
            for k in _FLAG_PTRS:
                trk[k] = o[k][:n]
        if q is not None:
            trk["cl_qcode"] = o["cl_qcode"][:n]
        if pos:            # O11: 16-bit integer positions, and residuals when the flags are on
            trk["cl_pos_code"] = o["cl_pos_code"][:n]
            if flags:
                trk["cl_res_code"] = o["cl_res_code"][:n]
        stg = {}
        if stages:
            for k in _STAGE_PTRS:
                stg[k] = o[k][:n] if k.startswith("link_") else o[k][:ns]
        return TrackResult(st, nt, nc, trk, stg)

    def status(self) -> tpcRunStatus:
        return tpcGetRunStatus(self.handle)

    def _host_buffers(self, capK, capC, slot):
        t = self.torch
        key = (capK, capC)
        bufs = getattr(self, "_host_slots", None)
        if bufs is None:
            bufs = self._host_slots = {}
        if slot not in bufs or bufs[slot][0] != key:
            def pinned(shape, dt, view=None):     # pinned host memory: the copies run asynchronously and at full speed
                a = t.empty(shape, dtype=dt, pin_memory=True).numpy()
                return a.view(view) if view is not None else a
            i32, f32 = t.int32, t.float32
            bufs[slot] = (key, {"trk_tracklet": pinned(capK, i32), "trk_sector": pinned(capK, i32),
                                "trk_first_row": pinned(capK, i32), "trk_last_row": pinned(capK, i32),
                                "trk_ncl": pinned(capK, i32), "trk_x": pinned(capK, f32), "trk_par": pinned((5, capK), f32),
                                "trk_cov": pinned((15, capK), f32), "trk_chi2": pinned(capK, f32),
                                "trk_cl_offset": pinned(capK + 1, i32, np.uint32),
                                "trk_cl_index": pinned(capC, i32, np.uint32)})
        return bufs[slot][1]

    def submit_host(self, slot: int, row_offset: np.ndarray, y: np.ndarray, z: np.ndarray, cap_tracks: int,
                    cap_track_clusters: int):
        """tpcSubmitHost: enqueue one event (host buffers, ideally pinned) on pipeline slot 0 or 1 and return at once."""
        L = load_library()
        n = int(y.shape[0])
        h = self._host_buffers(int(cap_tracks), int(cap_track_clusters), slot)
        tr = tpcTracks()
        tr.cap_tracks, tr.cap_track_clusters = int(cap_tracks), int(cap_track_clusters)
        for k, v in h.items():
            setattr(tr, k, v.ctypes.data)
        assert row_offset.dtype == np.uint32 and y.dtype == np.float32 and z.dtype == np.float32
        self._host_keep = getattr(self, "_host_keep", {})
        self._host_keep[slot] = (row_offset, y, z)          # the inputs must outlive the asynchronous copies
        rc = L.tpcSubmitHost(self.handle, slot, n, row_offset.ctypes.data, y.ctypes.data if n else None,
                             z.ctypes.data if n else None, byref(tr))
        if rc != TPC_OK:
            raise TpcError(rc, "tpcSubmitHost", L.tpcLastCudaError(self.handle).decode())

    def collect_host(self, slot: int):
        """tpcCollectHost: wait for the slot's event.  Returns (status, outputs); status.status may be TPC_ERR_CAPACITY
        (run that event again with run_host)."""
        L = load_library()
        st = tpcRunStatus()
        rc = L.tpcCollectHost(self.handle, slot, byref(st))
        if rc != TPC_OK:
            raise TpcError(rc, "tpcCollectHost", L.tpcLastCudaError(self.handle).decode())
        if st.status not in (TPC_OK, TPC_ERR_CAPACITY):
            raise TpcError(st.status, "tpcCollectHost (device status)")
        h = self._host_slots[slot][1]
        capK, capC = self._host_slots[slot][0]
        nt, nc = min(int(st.n_tracks), capK), min(int(st.n_track_clusters), capC)
        out = {k: (h[k][:, :nt] if h[k].ndim == 2 else h[k][:nt]) for k in _TRK_PTRS[:9]}
        out["trk_cl_offset"] = h["trk_cl_offset"][:nt + 1]
        out["trk_cl_index"] = h["trk_cl_index"][:nc]
        return st, out

    def run_host(self, row_offset: np.ndarray, y: np.ndarray, z: np.ndarray, cap_tracks: int | None = None,
                 cap_track_clusters: int | None = None):
        """tpcRunHost: host (numpy) buffers in, host buffers out; copies are part of the call."""
        L = load_library()
        n = int(y.shape[0])
        capK = int(cap_tracks) if cap_tracks is not None else max(4096, n // 8)
        capC = int(cap_track_clusters) if cap_track_clusters is not None else max(n, 1)
        key = (capK, capC)
        if getattr(self, "_host_key", None) != key:
            t = self.torch

            def pinned(shape, dt, view=None):     # pinned host memory: D2H copies run at full PCIe/C2C speed
                a = t.empty(shape, dtype=dt, pin_memory=True).numpy()
                return a.view(view) if view is not None else a
            i32, f32 = t.int32, t.float32
            self._host = {"trk_tracklet": pinned(capK, i32), "trk_sector": pinned(capK, i32),
                          "trk_first_row": pinned(capK, i32), "trk_last_row": pinned(capK, i32),
                          "trk_ncl": pinned(capK, i32), "trk_x": pinned(capK, f32), "trk_par": pinned((5, capK), f32),
                          "trk_cov": pinned((15, capK), f32), "trk_chi2": pinned(capK, f32),
                          "trk_cl_offset": pinned(capK + 1, i32, np.uint32), "trk_cl_index": pinned(capC, i32, np.uint32)}
            self._host_key = key
        tr = tpcTracks()
        tr.cap_tracks, tr.cap_track_clusters = capK, capC
        for k, v in self._host.items():
            setattr(tr, k, v.ctypes.data)
        st = tpcRunStatus()
        off = np.ascontiguousarray(row_offset, np.uint32)
        y = np.ascontiguousarray(y, np.float32)
        z = np.ascontiguousarray(z, np.float32)
        s = self.torch.cuda.current_stream(self.device).cuda_stream
        rc = L.tpcRunHost(self.handle, n, off.ctypes.data, y.ctypes.data if n else None, z.ctypes.data if n else None,
                          byref(tr), byref(st), s)
        if rc != TPC_OK:
            raise TpcError(rc, "tpcRunHost", L.tpcLastCudaError(self.handle).decode())
        if st.status not in (TPC_OK, TPC_ERR_CAPACITY):
            raise TpcError(st.status, "tpcRunHost (device status)")
        nt = min(int(st.n_tracks), capK)
        nc = min(int(st.n_track_clusters), capC)
        h = self._host
        out = {k: (h[k][:, :nt] if h[k].ndim == 2 else h[k][:nt]) for k in _TRK_PTRS[:9]}
        out["trk_cl_offset"] = h["trk_cl_offset"][:nt + 1]
        out["trk_cl_index"] = h["trk_cl_index"][:nc]
        return st, out
