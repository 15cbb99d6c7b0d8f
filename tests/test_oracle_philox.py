"""Pins of the oracle's random-number layer (no GPU).

* Philox4x32-10 against published known-answer vectors (tests/golden/philox4x32_10_kat.txt).
* The keyed call / uniform / offset / threshold helpers against the counter packing and bit-plane layout
  DESIGN.md §R3-R4 documents (convention — "parity unpinned" by any external source), assembled here
  from the KAT-pinned block function only.
* Statistical sanity of the streams (uniformity, fair offsets, independence of streams).
* "Is it still a fair 32-bit uniform": every one of the 32 bits of kpzref_uniform is fair and the bits are pairwise
  uncorrelated over 2^17 elements, U/2^32 passes a Kolmogorov-Smirnov test, acceptance frequencies of non-dyadic
  thresholds hold to 3 decimal places, and the nested-threshold property [U < 2^(32-k)] <=> "planes 0..k-1 are all zero"
  ties the plane ORDER to the sweep's acceptance rule (a zeroed, duplicated or swapped plane fails one of them).
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


# ------------------------------------------------------------------------------------------------------------------
# the uniform as a whole: all 32 planes (earlier pins only had power on planes 0-2)
# ------------------------------------------------------------------------------------------------------------------

_N_BITS = 1 << 17


@pytest.fixture(scope="module")
def uniforms():
    """U32 of 2^17 consecutive elements of three streams (PAIR pass 0, PAIR pass 1 at another time, SWITCH_AB)."""
    out = {}
    for name, (tag, tk, ps) in {"pair0": (R.TAGS["PAIR"], 7, 0), "pair1": (R.TAGS["PAIR"], (1 << 33) + 5, 1),
                                "switch": (R.TAGS["SWITCH_AB"], 123456, 0)}.items():
        out[name] = np.array([R.uniform(2024, tag, 3, tk, ps, e) for e in range(_N_BITS)], dtype=np.uint64)
    return out


@pytest.mark.parametrize("stream", ["pair0", "pair1", "switch"])
def test_every_bit_of_the_uniform_is_fair_and_bits_are_uncorrelated(uniforms, stream):
    u = uniforms[stream]
    n = len(u)
    bits = ((u[:, None] >> np.arange(32, dtype=np.uint64)[None, :]) & 1).astype(np.float64)      # [n][32]
    mean = bits.mean(axis=0)
    assert np.all(np.abs(mean - 0.5) < 5 * 0.5 / np.sqrt(n)), mean       # a stuck plane fails here
    c = np.corrcoef(bits.T)
    off = c[~np.eye(32, dtype=bool)]
    assert np.all(np.abs(off) < 5.5 / np.sqrt(n)), np.abs(off).max()     # a duplicated plane has correlation 1
    # neighbouring ELEMENTS are independent too (bit b of element e vs bit b of element e+1, e+32, e+128)
    for lag in (1, 32, 128):
        x, y = bits[:-lag], bits[lag:]
        r = ((x - 0.5) * (y - 0.5)).mean(axis=0) * 4
        assert np.all(np.abs(r) < 5 / np.sqrt(n - lag)), (lag, np.abs(r).max())


@pytest.mark.parametrize("stream", ["pair0", "pair1", "switch"])
def test_uniform_passes_kolmogorov_smirnov_and_hits_non_dyadic_thresholds(uniforms, stream):
    from scipy import stats
    u = uniforms[stream]
    n = len(u)
    x = (u.astype(np.float64) + 0.5) / 2.0**32
    assert stats.kstest(x, "uniform").pvalue > 1e-4
    # low 16 bits on their own (planes 16-31): a KS test of the high bits cannot see them
    lo = ((u & np.uint64(0xFFFF)).astype(np.float64) + 0.5) / 65536.0
    assert stats.kstest(lo, "uniform").pvalue > 1e-4
    for prob in (0.9, 0.1, 0.8, 0.3, 0.6, 0.05, 1.0 / 3.0):
        T = R.threshold(prob)
        f = (u < np.uint64(T)).mean()
        assert abs(f - T / 2.0**32) < 5 * np.sqrt(prob * (1 - prob) / n), (prob, f)


def test_plane_order_is_msb_first_through_the_acceptance_rule():
    """[U < 2^(32-k)] holds exactly when planes 0..k-1 of the element are all zero: plane b carries bit 31-b.  The
    left side is the acceptance rule of the sweep applied to kpzref_uniform, the right side comes from the
    KAT-pinned block function plane by plane; any permutation of the planes breaks the equivalence for some k."""
    seed, tag, sample, tk, ps = 99, R.TAGS["PAIR"], 1, 31, 0
    for element in (0, 5, 37, 127, 128, 1000, 4097):
        G, w, k = element >> 7, (element >> 5) & 3, element & 31
        plane_bits = [(R.philox_call(seed, tag, sample, tk, ps, b, G)[w] >> k) & 1 for b in range(32)]
        u = R.uniform(seed, tag, sample, tk, ps, element)
        for kk in range(1, 33):
            assert (u < (1 << (32 - kk))) == (not any(plane_bits[:kk]))
