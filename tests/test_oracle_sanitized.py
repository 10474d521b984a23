"""The oracle under AddressSanitizer and UndefinedBehaviorSanitizer: the same source, built with -fsanitize=address,undefined
and the oracle's own arithmetic flags, runs every stage (O1..O12) on small seeded events in a fresh process, and its results
equal those of the normal build.  The oracle is the yardstick of every parity test: an out-of-bounds read or an
uninitialised value in it would be compared against, not found.  CPU only."""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "tpc_oracle.cpp")

CODE = r"""
import hashlib, sys
import numpy as np
sys.path.insert(0, %r)
from oracle import tpc_oracle as orc
from paper_1910_12214_b200 import datagen
h = hashlib.sha256()
for idx, scale, dead in ((0, 1.0, ()), (1, 0.03, (30, 31)), (2, 0.06, ()), (3, 0.004, (100,))):
    ev = datagen.make_event(idx, scale=scale, dead_rows=dead)
    r = orc.run(ev, merged=True, flags=True)
    for a in (r.link_up, r.link_dn, r.start_hits, r.tl_status, r.tl_rowhit, r.trk_cl_index, r.trk_par, r.trk_cov, r.mg_next,
              r.lg_partner, r.mt_id, r.mt_cl_index, r.cf_flags, r.cf_owner):
        h.update(np.ascontiguousarray(a).tobytes())
    b = orc.run(ev, brute_force=True)                 # the brute-force searches of the pins
    h.update(np.ascontiguousarray(b.trk_cl_index).tobytes())
print("DIGEST", h.hexdigest())
""" % ROOT


def _run(env_extra):
    env = dict(os.environ)
    env.update(env_extra)
    p = subprocess.run([sys.executable, "-c", CODE], capture_output=True, text=True, env=env, timeout=900)
    return p


@pytest.mark.skipif(shutil.which("g++") is None, reason="g++ not available")
def test_oracle_is_clean_under_asan_and_ubsan_and_gives_the_same_results(tmp_path):
    so = str(tmp_path / "libtpcoracle_san.so")
    subprocess.check_call(["g++", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                           "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", SRC, "-o", so])
    libasan = subprocess.check_output(["g++", "-print-file-name=libasan.so"], text=True).strip()
    if not os.path.isabs(libasan) or not os.path.exists(libasan):
        pytest.skip("libasan.so not found")
    plain = _run({})
    assert plain.returncode == 0, plain.stderr[-2000:]
    san = _run({"TPC_ORACLE_LIB": so, "LD_PRELOAD": libasan, "ASAN_OPTIONS": "detect_leaks=0:abort_on_error=0",
                "UBSAN_OPTIONS": "print_stacktrace=1"})
    assert san.returncode == 0, san.stderr[-3000:]
    assert "AddressSanitizer" not in san.stderr and "runtime error" not in san.stderr, san.stderr[-3000:]
    d0 = [l for l in plain.stdout.splitlines() if l.startswith("DIGEST")]
    d1 = [l for l in san.stdout.splitlines() if l.startswith("DIGEST")]
    assert d0 and d0 == d1          # -O1 with the sanitizers against -O2 without: the same bits (no FMA, no reassociation)
