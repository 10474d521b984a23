"""CPU-only checks of the boundary: libtpcgpu.so builds, loads and exports every symbol include/tpc_abi.h declares;
host-side argument logic that needs no device.  No compute call is made here."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1910_12214_b200 import tpc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "tpc_abi.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tpc[A-Z]\w*)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    lib = tpc.load_library()
    names = _declared_functions()
    assert set(names) == set(tpc.ABI_SYMBOLS), (names, tpc.ABI_SYMBOLS)
    for n in names:
        assert getattr(lib, n) is not None


def test_struct_layouts_match_the_header():
    """sizeof of the ctypes mirrors == sizeof in C (compiled from the header with the host compiler)."""
    import subprocess
    import tempfile
    code = '#include "tpc_abi.h"\n#include <stdio.h>\nint main(){printf("%zu %zu %zu %zu %zu\\n",sizeof(tpcGeometry),' \
           'sizeof(tpcParams),sizeof(tpcClusters),sizeof(tpcTracks),sizeof(tpcRunStatus));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write(code)
        exe = os.path.join(d, "s")
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe])
        sizes = [int(x) for x in subprocess.check_output([exe]).split()]
    mine = [ctypes.sizeof(t) for t in (tpc.tpcGeometry, tpc.tpcParams, tpc.tpcClusters, tpc.tpcTracks, tpc.tpcRunStatus)]
    assert sizes == mine


def test_default_params_are_table_p():
    p = tpc.tpcDefaultParams()
    want = dict(area_y=1.5, area_z=1.5, link_dev2_max=0.64, err2_y=0.01, err2_z=0.01, init_var_s=1.0, init_var_t=1.0,
                init_var_q=100.0, turn_var_scale=100.0, max_sinphi=0.98, road_sigma=4.0, road_min=0.3, road_max=2.0,
                max_row_gap=4, min_chain_hits=3, min_tracklet_hits=10, min_track_hits=10, cell_min=0.5, cell_max=8.0)
    for k, v in want.items():
        assert getattr(p, k) == pytest.approx(v, rel=1e-7), k
    # the oracle's own defaults are the same table (two independent copies of Table P)
    from oracle import tpc_oracle as orc
    o = orc.default_params()
    for k in want:
        assert getattr(o, k) == getattr(p, k), k


def test_error_strings_and_argument_checks_without_a_device():
    lib = tpc.load_library()
    for code in (0, -1, -2, -3, -4, -5, -6, -7, -8):
        assert len(lib.tpcErrorString(code)) > 1 and lib.tpcErrorString(code) != lib.tpcErrorString(-99)
    assert lib.tpcDefaultParams(None) == tpc.TPC_ERR_INVALID_ARG
    h = ctypes.c_void_p()
    p = tpc.tpcDefaultParams()
    row_x = np.linspace(85, 245, 152).astype(np.float32)
    g = tpc.tpcGeometry(36, 152, row_x.ctypes.data, None, None, 0.5, 0.176, -250.0, 250.0)
    assert lib.tpcCreate(ctypes.byref(h), None, ctypes.byref(p), 0) == tpc.TPC_ERR_INVALID_ARG
    bad = tpc.tpcGeometry(36, 2, row_x.ctypes.data, None, None, 0.5, 0.176, -250.0, 250.0)      # n_rows < 3
    assert lib.tpcCreate(ctypes.byref(h), ctypes.byref(bad), ctypes.byref(p), 0) == tpc.TPC_ERR_INVALID_ARG
    bad = tpc.tpcGeometry(65, 152, row_x.ctypes.data, None, None, 0.5, 0.176, -250.0, 250.0)    # n_sectors > 64 (header)
    assert lib.tpcCreate(ctypes.byref(h), ctypes.byref(bad), ctypes.byref(p), 0) == tpc.TPC_ERR_INVALID_ARG
    # the allocation-free entry point checks its arguments before it touches the device
    assert lib.tpcNoAllocMaxClusters() == 1 << 24
    assert lib.tpcStartHitsNoAlloc(0, (1 << 24) + 1, 8, 8, 8, 1, 8, None) == tpc.TPC_ERR_NOALLOC_LIMIT
    assert b"TPC_NOALLOC_MAX_CLUSTERS" in lib.tpcNoAllocLastError()
    assert lib.tpcStartHitsNoAlloc(0, 10, None, 8, 8, 1, 8, None) == tpc.TPC_ERR_INVALID_ARG
    assert lib.tpcStartHitsNoAlloc(0, -1, 8, 8, 8, 1, 8, None) == tpc.TPC_ERR_INVALID_ARG
    assert lib.tpcNoAllocSetup(-1) == tpc.TPC_ERR_INVALID_ARG
    rev = row_x[::-1].copy()                                                                     # not increasing
    bad = tpc.tpcGeometry(36, 152, rev.ctypes.data, None, None, 0.5, 0.176, -250.0, 250.0)
    assert lib.tpcCreate(ctypes.byref(h), ctypes.byref(bad), ctypes.byref(p), 0) == tpc.TPC_ERR_INVALID_ARG
    import torch
    if not torch.cuda.is_available():
        # no device: creation fails loudly with TPC_ERR_CUDA -- there is no CPU fallback behind the ABI
        assert lib.tpcCreate(ctypes.byref(h), ctypes.byref(g), ctypes.byref(p), 0) == tpc.TPC_ERR_CUDA
        with pytest.raises(RuntimeError):
            tpc.TpcTracker(36, 152, row_x)


def test_product_path_does_not_import_the_oracle():
    """The package never imports oracle/ (only tests, smoke() and bench.py's cpu_baseline legs may)."""
    pkg = os.path.join(ROOT, "paper_1910_12214_b200")
    pat = re.compile(r"(^|\n)\s*(import|from)\s+oracle|#include\s+[\"<][^\n]*oracle|libtpcoracle|tpc_oracle\.(py|h|cpp)|orcRun")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not pat.search(txt), os.path.join(dirpath, f)
