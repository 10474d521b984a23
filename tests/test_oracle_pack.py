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
