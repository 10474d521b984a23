"""Seeded synthetic TPC cluster inputs (BASELINE.json configs 0-4).

This module serves both the oracle tests and the CUDA path.  It contains no tracker arithmetic; it
wraps ``tpcgen.cpp`` (helix / pad-row-plane intersections, smearing, shuffling) through ctypes and
names the five workloads.  The data stand in for the ALICE pp event and the simulated Pb-Pb
collisions the paper measures on (Fig. 4, L106 Fig. 6), which are not available.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpcgen.cpp")
_LIB = os.path.join(_HERE, "libtpcgen.so")

N_ROWS = 152
TAN_HALF_SECTOR = math.tan(math.radians(10.0))
BZ_TESLA = 0.5
Z_ABS_MAX = 250.0


def default_row_x(n_rows: int = N_ROWS) -> np.ndarray:
    """x_r = 85 + r*160/151 cm ('152 pad rows at radii 85-245 cm')."""
    r = np.arange(n_rows, dtype=np.float64)
    return 85.0 + r * (160.0 / (n_rows - 1))


def default_row_pitch(n_rows: int = N_ROWS) -> np.ndarray:
    """0.4 cm for r < 63, 0.6 cm above; carried, not used by the tracking arithmetic."""
    return np.where(np.arange(n_rows) < 63, 0.4, 0.6).astype(np.float32)


def build(force: bool = False) -> str:
    """Compile libtpcgen.so in-tree (g++, seconds)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-shared", "-fPIC", "-fopenmp", _SRC, "-o", _LIB])
    return _LIB


class _Population(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int32), ("max_turns", ctypes.c_int32), ("n_tracks", ctypes.c_int64),
                ("pt_lo", ctypes.c_double), ("pt_hi", ctypes.c_double), ("pt_scale", ctypes.c_double),
                ("phi_lo", ctypes.c_double), ("phi_hi", ctypes.c_double), ("eta_max", ctypes.c_double)]


class _Config(ctypes.Structure):
    _fields_ = [("seed", ctypes.c_uint64), ("n_sectors", ctypes.c_int32), ("n_rows", ctypes.c_int32),
                ("row_x", ctypes.POINTER(ctypes.c_double)), ("bz_tesla", ctypes.c_double),
                ("tan_half_sector", ctypes.c_double), ("z_abs_max", ctypes.c_double),
                ("sigma_y", ctypes.c_double), ("sigma_z", ctypes.c_double), ("noise_frac", ctypes.c_double),
                ("vtx_sigma_z", ctypes.c_double), ("n_collisions", ctypes.c_int32), ("n_pop", ctypes.c_int32),
                ("pop", ctypes.POINTER(_Population)), ("mult_mean", ctypes.c_double), ("mult_cap", ctypes.c_double),
                ("t0_window_us", ctypes.c_double), ("v_drift_cm_per_us", ctypes.c_double)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        lib.tpcgen_generate.restype = ctypes.c_void_p
        lib.tpcgen_generate.argtypes = [ctypes.POINTER(_Config)]
        lib.tpcgen_n_clusters.restype = ctypes.c_int64
        lib.tpcgen_n_clusters.argtypes = [ctypes.c_void_p]
        lib.tpcgen_n_tracks.restype = ctypes.c_int64
        lib.tpcgen_n_tracks.argtypes = [ctypes.c_void_p]
        lib.tpcgen_copy_clusters.restype = None
        lib.tpcgen_copy_clusters.argtypes = [ctypes.c_void_p] * 8
        lib.tpcgen_copy_tracks.restype = None
        lib.tpcgen_copy_tracks.argtypes = [ctypes.c_void_p] * 7
        lib.tpcgen_free.restype = None
        lib.tpcgen_free.argtypes = [ctypes.c_void_p]
        _lib = lib
    return _lib


@dataclass
class Population:
    kind: int            # 0 log-uniform, 1 pT*exp(-pT/scale), 2 uniform
    n_tracks: int
    pt_lo: float
    pt_hi: float
    pt_scale: float = 0.3
    phi_lo: float = 0.0
    phi_hi: float = 2.0 * math.pi
    eta_max: float = 0.9
    max_turns: int = 1


@dataclass
class GenConfig:
    seed: int
    n_sectors: int
    populations: list
    noise_frac: float = 0.0
    vtx_sigma_z: float = 0.0
    n_collisions: int = 1
    mult_mean: float = 2000.0
    mult_cap: float = 8000.0
    t0_window_us: float = 100.0
    v_drift_cm_per_us: float = 2.5
    sigma_y: float = 0.1
    sigma_z: float = 0.1
    n_rows: int = N_ROWS
    bz_tesla: float = BZ_TESLA
    row_x: np.ndarray = field(default_factory=default_row_x)
    dead_rows: tuple = ()


@dataclass
class Event:
    """Host-side (numpy) clusters, CSR by (sector,row), fp32 SoA, plus geometry and generator truth."""
    n_sectors: int
    n_rows: int
    row_x: np.ndarray          # float32 [n_rows]
    row_pitch: np.ndarray      # float32 [n_rows]
    row_dead: np.ndarray       # uint8 [n_rows]
    bz_tesla: float
    tan_half_sector: float
    z_min: float
    z_max: float
    row_offset: np.ndarray     # uint32 [n_sectors*n_rows+1]
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    q: np.ndarray
    truth_track: np.ndarray    # int32 [n_clusters], -1 = noise
    truth_turn: np.ndarray
    trk_pt: np.ndarray         # float64 [n_gen_tracks]
    trk_phi0: np.ndarray
    trk_eta: np.ndarray
    trk_vz: np.ndarray
    trk_zshift: np.ndarray
    trk_h: np.ndarray          # int32: direction angle = phi0 - h*psi
    name: str = ""

    @property
    def n_clusters(self) -> int:
        return int(self.y.shape[0])


def generate(cfg: GenConfig, name: str = "") -> Event:
    lib = _load()
    row_x = np.ascontiguousarray(cfg.row_x, dtype=np.float64)
    pops = (_Population * len(cfg.populations))()
    for i, p in enumerate(cfg.populations):
        pops[i] = _Population(p.kind, p.max_turns, p.n_tracks, p.pt_lo, p.pt_hi, p.pt_scale, p.phi_lo, p.phi_hi,
                              p.eta_max)
    c = _Config(cfg.seed, cfg.n_sectors, cfg.n_rows, row_x.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                cfg.bz_tesla, TAN_HALF_SECTOR, Z_ABS_MAX, cfg.sigma_y, cfg.sigma_z, cfg.noise_frac, cfg.vtx_sigma_z,
                cfg.n_collisions, len(cfg.populations), pops, cfg.mult_mean, cfg.mult_cap, cfg.t0_window_us,
                cfg.v_drift_cm_per_us)
    h = lib.tpcgen_generate(ctypes.byref(c))
    if not h:
        raise ValueError("tpcgen_generate rejected the configuration")
    try:
        n = lib.tpcgen_n_clusters(h)
        nt = lib.tpcgen_n_tracks(h)
        ro = np.empty(cfg.n_sectors * cfg.n_rows + 1, np.uint32)
        x, y, z, q = (np.empty(n, np.float32) for _ in range(4))
        tt, tu = np.empty(n, np.int32), np.empty(n, np.int32)
        lib.tpcgen_copy_clusters(h, ro.ctypes.data, x.ctypes.data, y.ctypes.data, z.ctypes.data, q.ctypes.data,
                                 tt.ctypes.data, tu.ctypes.data)
        pt, phi0, eta, vz, zs = (np.empty(nt, np.float64) for _ in range(5))
        hs = np.empty(nt, np.int32)
        lib.tpcgen_copy_tracks(h, pt.ctypes.data, phi0.ctypes.data, eta.ctypes.data, vz.ctypes.data, zs.ctypes.data,
                               hs.ctypes.data)
    finally:
        lib.tpcgen_free(h)
    dead = np.zeros(cfg.n_rows, np.uint8)
    for r in cfg.dead_rows:
        dead[r] = 1
    if dead.any():
        # clusters on dead rows are removed (a dead row delivers no data)
        keep = np.ones(n, bool)
        counts = np.diff(ro.astype(np.int64))
        for s in range(cfg.n_sectors):
            for r in cfg.dead_rows:
                b = s * cfg.n_rows + r
                keep[ro[b]:ro[b + 1]] = False
                counts[b] = 0
        x, y, z, q, tt, tu = (a[keep] for a in (x, y, z, q, tt, tu))
        ro = np.concatenate([[0], np.cumsum(counts)]).astype(np.uint32)
    # the grid z range is the whole drift range on both signs for every config
    return Event(cfg.n_sectors, cfg.n_rows, row_x.astype(np.float32), default_row_pitch(cfg.n_rows), dead,
                 cfg.bz_tesla, TAN_HALF_SECTOR, -Z_ABS_MAX, Z_ABS_MAX, ro, x, y, z, q, tt, tu,
                 pt, phi0, eta, vz, zs, hs, name)


_SPECTRUM = dict(kind=1, pt_lo=0.1, pt_hi=20.0, pt_scale=0.3)


def config(idx: int, scale: float = 1.0, seed: int | None = None, dead_rows: tuple = ()) -> GenConfig:
    """The five workloads of BASELINE.json (`configs[idx]`); seeds 1..5.

    ``scale`` shrinks the track / collision counts proportionally (for bounded CPU samples); 1.0 is
    the configuration as named.
    """
    s = (idx + 1) if seed is None else seed
    if idx == 0:
        a = math.radians(10.0)
        return GenConfig(s, 1, [Population(0, max(1, round(200 * scale)), 0.2, 10.0, phi_lo=a - math.radians(10.0),
                                           phi_hi=a + math.radians(10.0))], dead_rows=dead_rows)
    if idx == 1:
        return GenConfig(s, 36, [Population(n_tracks=max(1, round(8000 * scale)), **_SPECTRUM)], noise_frac=0.05,
                         vtx_sigma_z=5.0, dead_rows=dead_rows)
    if idx == 2:
        return GenConfig(s, 36, [Population(2, max(1, round(2000 * scale)), 0.05, 0.15, max_turns=2),
                                 Population(n_tracks=max(1, round(4000 * scale)), **_SPECTRUM)], noise_frac=0.10,
                         vtx_sigma_z=5.0, dead_rows=dead_rows)
    if idx in (3, 4):
        ncoll = 50 if idx == 3 else 200
        return GenConfig(s, 36, [Population(n_tracks=0, **_SPECTRUM)], noise_frac=0.05, vtx_sigma_z=5.0,
                         n_collisions=max(2, round(ncoll * scale)), dead_rows=dead_rows)
    raise ValueError(f"no config {idx}")


def make_event(idx: int, scale: float = 1.0, seed: int | None = None, dead_rows: tuple = ()) -> Event:
    return generate(config(idx, scale, seed, dead_rows), name=f"config{idx}" + ("" if scale == 1.0 else f"@{scale:g}"))


def event_from_arrays(row_offset, y, z, n_sectors: int, n_rows: int, row_x=None, row_dead=None, z_min=-Z_ABS_MAX,
                      z_max=Z_ABS_MAX, bz_tesla=BZ_TESLA) -> Event:
    """Wrap hand-built clusters (tests) in an Event."""
    row_x = default_row_x(n_rows).astype(np.float32) if row_x is None else np.asarray(row_x, np.float32)
    row_offset = np.asarray(row_offset, np.uint32)
    y = np.asarray(y, np.float32)
    z = np.asarray(z, np.float32)
    n = y.shape[0]
    counts = np.diff(row_offset.astype(np.int64))
    rows = np.repeat(np.arange(n_sectors * n_rows) % n_rows, counts)
    x = row_x[rows].astype(np.float32) if n else np.zeros(0, np.float32)
    dead = np.zeros(n_rows, np.uint8) if row_dead is None else np.asarray(row_dead, np.uint8)
    e = np.zeros(0, np.float64)
    return Event(n_sectors, n_rows, row_x, default_row_pitch(n_rows), dead, bz_tesla, TAN_HALF_SECTOR, z_min, z_max,
                 row_offset, x, y, z, np.ones(n, np.float32), np.full(n, -1, np.int32), np.full(n, -1, np.int32),
                 e, e, e, e, e, np.zeros(0, np.int32), "custom")
