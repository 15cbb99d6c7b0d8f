"""Pins of the oracle's random-number layer (no GPU).

* Philox4x32-10 against published known-answer vectors (tests/golden/philox4x32_10_kat.txt).
* The keyed call / uniform / offset / threshold helpers against the counter packing and bit-plane layout
  DESIGN.md §R3-R4 documents (convention — "parity unpinned" by any external source), assembled here
  from the KAT-pinned block function only.
* Statistical sanity of the streams (uniformity, fair offsets, independence of streams).
"""
import os

import numpy as np
import pytest

from oracle import kpzref as R

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _kat():
    rows = []
    with open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            v = [int(x, 16) for x in line.split()]
            rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_philox_known_answers():
    rows = _kat()
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert R.philox4x32_10(ctr, key) == out


def test_philox_is_a_bijection_of_the_counter_for_fixed_key():
    # distinct counters -> distinct outputs (Philox is a keyed permutation of the 128-bit counter)
    outs = {tuple(R.philox4x32_10([c, 0, 0, 0], [1, 2])) for c in range(2000)}
    assert len(outs) == 2000


@pytest.mark.parametrize("seed,tag,sample,timekey,pass_,plane,G", [
    (1, 0, 0, 0, 0, 0, 0),
    (0x0123456789ABCDEF, 1, 7, 999, 1, 0, 0),
    (5, 9, 255, (1 << 40) + 12345, 0, 31, 77),
    (2, 6, 1023, (1 << 54) - 1, 1, 17, 0xFFFFFFFF),
])
def test_keyed_call_uses_documented_counter_packing(seed, tag, sample, timekey, pass_, plane, G):
    # c0=G, c1=sample, c2=timekey low, c3 = tag<<28 | pass<<27 | plane<<22 | timekey>>32; key = seed lo, hi
    ctr = [G, sample, timekey & 0xFFFFFFFF, (tag << 28) | (pass_ << 27) | (plane << 22) | (timekey >> 32)]
    key = [seed & 0xFFFFFFFF, seed >> 32]
    assert R.philox_call(seed, tag, sample, timekey, pass_, plane, G) == R.philox4x32_10(ctr, key)


def test_keyed_call_rejects_out_of_range_fields():
    with pytest.raises(R.OracleError):
        R.philox_call(1, 16, 0, 0, 0, 0, 0)
    with pytest.raises(R.OracleError):
        R.philox_call(1, 0, 0, 1 << 54, 0, 0, 0)
    with pytest.raises(R.OracleError):
        R.philox_call(1, 0, 0, 0, 2, 0, 0)
    with pytest.raises(R.OracleError):
        R.philox_call(1, 0, 0, 0, 0, 32, 0)


@pytest.mark.parametrize("element", [0, 1, 31, 32, 127, 128, 4095, 123457])
def test_uniform_is_msb_first_bit_plane_assembly(element):
    seed, tag, sample, tk, ps = 11, 0, 3, 42, 1
    G, w, k = element >> 7, (element >> 5) & 3, element & 31
    u = 0
    for b in range(32):
        u |= ((R.philox_call(seed, tag, sample, tk, ps, b, G)[w] >> k) & 1) << (31 - b)
    assert R.uniform(seed, tag, sample, tk, ps, element) == u


def test_threshold_values():
    assert R.threshold(0.0) == 0
    assert R.threshold(1.0) == 1 << 32
    assert R.threshold(0.5) == 0x80000000
    assert R.threshold(0.75) == 0xC0000000
    assert R.threshold(0.25) == 0x40000000
    assert R.threshold(0.9) == 0xE6666666     # floor(0.9 * 2^32), 0.9 as the nearest double
    assert R.threshold(0.1) == 0x19999999
    assert R.threshold(0.05) == 0x0CCCCCCC
    assert R.threshold(0.3) == 0x4CCCCCCC
    for bad in (-0.1, 1.0000001, float("nan")):
        with pytest.raises(R.OracleError):
            R.threshold(bad)


def test_offset_is_bit0_of_word0_of_the_offset_stream():
    for sample, m, ps in [(0, 0, 0), (5, 17, 1), (1023, 10**9, 0)]:
        w = R.philox_call(9, R.TAGS["OFFSET"], sample, m, ps, 0, 0)
        assert R.offset(9, sample, m, ps) == (w[0] & 1)


def test_offsets_are_a_fair_coin():
    n = 20000
    ones = sum(R.offset(123, s % 8, m, ps) for s, (m, ps) in enumerate((i // 2, i % 2) for i in range(n)))
    # binomial(n, 1/2): sigma = sqrt(n)/2
    assert abs(ones - n / 2) < 5 * np.sqrt(n) / 2


def test_uniforms_are_uniform_and_streams_differ():
    n = 3000
    u0 = np.array([R.uniform(77, R.TAGS["PAIR"], 0, 5, 0, e) for e in range(n)], dtype=np.float64) / 2.0**32
    u1 = np.array([R.uniform(77, R.TAGS["PAIR"], 0, 5, 1, e) for e in range(n)], dtype=np.float64) / 2.0**32
    u2 = np.array([R.uniform(77, R.TAGS["PAIR_B"], 0, 5, 0, e) for e in range(n)], dtype=np.float64) / 2.0**32
    for u in (u0, u1, u2):
        assert abs(u.mean() - 0.5) < 5 * np.sqrt(1 / 12 / n)
        assert abs((u < 0.9).mean() - 0.9) < 5 * np.sqrt(0.09 / n)
        assert abs((u < 0.25).mean() - 0.25) < 5 * np.sqrt(0.1875 / n)
    # streams (pass, tag) are different sequences and uncorrelated
    assert not np.array_equal(u0, u1) and not np.array_equal(u0, u2)
    for a, b in ((u0, u1), (u0, u2)):
        assert abs(np.corrcoef(a, b)[0, 1]) < 5 / np.sqrt(n)
