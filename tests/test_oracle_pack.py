"""Pins of the oracle's O9 dynamic-precision charge code (DESIGN.md section 3 "O9", reading R38).

The paper's sentence is a definition: every bit more than n after the first non-zero bit is rounded away.  Brute force
over ALL 16-bit values and n = 1..6 against a definition written independently here: the representable codes are the
integers with at most n+1 significant bits, and the code of v is the representable value nearest to v (ties up).
"""
import numpy as np
import pytest

from oracle import tpc_oracle as orc


def _representable(n):
    vals = {0}
    for top in range(16):                       # position of the leading one
        for m in range(1 << min(top, n)):       # the up to n bits right after it
            vals.add((1 << top) | (m << max(top - n, 0)) if top >= n else (1 << top) | m)
    return np.array(sorted(v for v in vals if v <= 65535), np.int64)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6])
def test_code_is_the_nearest_value_with_n_plus_one_significant_bits_for_every_16_bit_input(n):
    v = np.arange(65536, dtype=np.int64)
    code = orc.pack_charge(v.astype(np.float32), n).astype(np.int64)
    rep = _representable(n)
    assert np.all(np.isin(code, rep))                                   # at most n+1 significant bits
    # nearest representable value, ties to the upper one, by brute force over the representable set
    idx = np.searchsorted(rep, v)
    lo = rep[np.maximum(idx - 1, 0)]
    hi = rep[np.minimum(idx, len(rep) - 1)]
    want = np.where(v - lo < hi - v, lo, hi)
    want = np.where(np.isin(v, rep), v, want)
    want = np.minimum(want, rep[-1])                                    # saturation at the largest code
    assert np.array_equal(code, want)
    # the paper's wording, bit by bit: small values are exact, the relative error is bounded by 2^-(n+1)
    assert np.array_equal(code[: 1 << (n + 1)], v[: 1 << (n + 1)])
    ok = v <= rep[-1]
    assert np.all(np.abs(code[ok] - v[ok]) * (1 << (n + 1)) <= np.maximum(v[ok], 1))
    assert np.all(np.diff(code) >= 0)                                   # monotone
    assert np.array_equal(orc.pack_charge(code.astype(np.float32), n).astype(np.int64), code)      # idempotent


def test_float_inputs_round_to_the_nearest_integer_first_and_bad_values_are_clamped():
    q = np.array([0.0, 0.49, 0.5, 1.5, 2.5, 31.49, 31.5, 33.0, 99.99, -3.0, np.nan, 1e9, 65535.0], np.float32)
    code = orc.pack_charge(q, 4)
    #              0   0    0(even) 2   2     31     32    34->? 100->?  0    0   sat   sat
    assert list(code[:7]) == [0, 0, 0, 2, 2, 31, 32]
    assert code[7] == 34 and code[8] == 100          # 33 = 100001b -> 6 bits, keep 5: 34 (tie up); 100 = 1100100b -> 100
    assert code[9] == 0 and code[10] == 0 and code[11] == 63488 and code[12] == 63488
    assert list(orc.pack_charge(np.array([33.0, 100.0, 1000.0], np.float32), 3)) == [32, 104, 1024]


def _golden():
    import os
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "charge_codes.txt")) if l[0] != "#"]
    a = np.array(rows, np.float64)
    return a[:, 0].astype(np.float32), a[:, 1].astype(np.uint16), a[:, 2].astype(np.uint16)


def test_golden_charge_codes_and_a_few_values_worked_by_hand():
    q, c4, c3 = _golden()
    assert np.array_equal(orc.pack_charge(q, 4), c4) and np.array_equal(orc.pack_charge(q, 3), c3)
    # worked by hand from the sentence of PAPER.md L70: 67 = 1000011b, n = 4 keeps 10000|11 -> rounds up to 1000100b = 68;
    # 1000 = 1111101000b, n = 4 keeps 11111|01000 -> 1111100000b = 992;  n = 3 keeps 1111|101000 -> rounds up to 1024
    d = {float(v): (int(a), int(b)) for v, a, b in zip(q, c4, c3)}
    assert d[67.0] == (68, 64) and d[1000.0] == (992, 1024) and d[35.0] == (36, 36) and d[17.0] == (17, 18)


# ---- O11: 16-bit integer format of positions and residuals (rest of NEXT-4; DESIGN.md section 3 "O11", R45) -----------
def _unpack(code):
    c = np.asarray(code, np.uint32)
    return (c & 0xFFFF).astype(np.uint16).view(np.int16).astype(np.int64), (c >> 16).astype(np.uint16).view(np.int16).astype(np.int64)


@pytest.mark.parametrize("bits", [0, 4, 6, 8])
def test_position_code_is_the_nearest_lattice_point(bits):
    rng = np.random.default_rng(50 + bits)
    q = 2.0 ** -bits
    lim = 32767 * q
    y = rng.uniform(-min(lim, 250.0), min(lim, 250.0), 200000).astype(np.float32)
    z = rng.uniform(-min(lim, 250.0), min(lim, 250.0), 200000).astype(np.float32)
    cy, cz = _unpack(orc.pack_positions(y, z, bits))
    for v, c in ((y, cy), (z, cz)):
        v64 = v.astype(np.float64)
        assert np.all(np.abs(c * q - v64) <= q / 2)                      # nearest lattice point: error at most half a unit
        assert np.array_equal(c, np.rint(v64 / q).astype(np.int64))        # numpy's rint is ties-to-even too
    # lattice points are exact and the code is monotone
    k = np.arange(-32768, 32768, dtype=np.int64)
    ck, _ = _unpack(orc.pack_positions((k * q).astype(np.float32), np.zeros(len(k), np.float32), bits))
    assert np.array_equal(ck, k)
    s = np.sort(y)
    assert np.all(np.diff(_unpack(orc.pack_positions(s, s, bits))[0]) >= 0)


def test_position_code_ties_saturation_and_bad_values_by_hand():
    # units of 1/64 cm: 0.5/64 -> tie -> 0 (even); 1.5/64 -> 2; 2.5/64 -> 2; -0.5/64 -> 0; -1.5/64 -> -2
    y = np.array([0.5, 1.5, 2.5, -0.5, -1.5, 64.0, 1e9, -1e9, np.nan, np.inf, -np.inf, 511.984375, 512.0], np.float64) / 64.0
    y[5] = 1.0                                   # exactly 64 units
    y[6:11] = [1e9, -1e9, np.nan, np.inf, -np.inf]
    y[11], y[12] = 32767.0 / 64.0, 32768.0 / 64.0
    cy, cz = _unpack(orc.pack_positions(y.astype(np.float32), (-y).astype(np.float32), 6))
    assert list(cy) == [0, 2, 2, 0, -2, 64, 32767, -32768, 0, 32767, -32768, 32767, 32767]
    assert list(cz) == [0, -2, -2, 0, 2, -64, -32768, 32767, 0, -32768, 32767, -32767, -32768]
    with pytest.raises(ValueError):
        orc.pack_positions(np.zeros(2, np.float32), np.zeros(2, np.float32), 16)


def test_residual_codes_of_a_run_are_the_packed_residuals_and_cost_less_than_a_percent_of_the_resolution():
    from paper_1910_12214_b200 import datagen
    ev = datagen.make_event(0)
    res = orc.run(ev, flags=True)
    cy, cz = _unpack(res.cf_res_code)
    assert np.array_equal(cy, np.rint(res.cf_res_y * 64).astype(np.int64)) and np.array_equal(cz, np.rint(res.cf_res_z * 64).astype(np.int64))
    att = res.cf_res_y != 0
    assert att.sum() > 8000 and np.all(cy[~att] == 0)
    # quantisation noise q / sqrt(12) = 0.0045 cm against the 0.1 cm resolution of config 0: the variance grows by 0.2 %
    err = cy[att] / 64.0 - res.cf_res_y[att]
    assert np.std(err) == pytest.approx(2.0 ** -6 / np.sqrt(12.0), rel=0.05)
    assert np.var(cy[att] / 64.0) < 1.01 * np.var(res.cf_res_y[att])
    # 16 bits are far more than the residuals need: they fit 7 bits (the entropy coder's business, out of scope)
    assert np.abs(cy[att]).max() < 64 and np.abs(cz[att]).max() < 64
