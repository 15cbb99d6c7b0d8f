"""Host-side analysis helpers (paper_1012_0385_b200/analysis.py) against exact arithmetic, synthetic scaling forms and
the oracle."""
from fractions import Fraction

import numpy as np

from oracle import kpzref as R
from paper_1012_0385_b200 import analysis as A


def test_w2_matches_exact_fractions_and_the_oracle_mean():
    L, S = 256, 5
    sim = R.KpzRef(L, S, 0.75, 0.25, seed=3)
    sim.set_record_times([1, 9, 40])
    sim.run(40)
    r = sim.roughness()
    w2 = A.w2_per_sample(L, r["sum_h"], r["sum_h2"])
    for k in range(3):
        for s in range(S):
            exact = Fraction(L * int(r["sum_h2"][k, s]) - int(r["sum_h"][k, s]) ** 2, L * L)
            assert abs(w2[k, s] - float(exact)) <= 1e-15 * max(1.0, float(exact))
    assert np.allclose(A.w2_mean(L, r["sum_h"], r["sum_h2"]), r["w2_mean"], rtol=1e-15, atol=0)
    # sums beyond 64 bits in the numerator do not overflow
    big = A.w2_per_sample(1 << 28, np.array([[3 << 40]]), np.array([[7 << 58]]))
    assert big[0, 0] == float(Fraction((1 << 28) * (7 << 58) - (3 << 40) ** 2, 1 << 56))


def test_exponents_on_power_laws_and_collapse_of_a_scaling_form():
    t = np.array([2.0 ** k for k in range(1, 14)])
    w2 = 0.25 + 0.7 * t ** (2.0 / 3.0)
    assert np.allclose(A.local_exponents(t, w2 - 0.25), 2.0 / 3.0)
    assert abs(A.growth_exponent(t, w2) - 1.0 / 3.0) < 1e-12
    # W^2 - 1/4 = L^(2 alpha) f(t / L^z) with f(x) = x^(2 beta) / (1 + x^(2 beta)): a perfect collapse with (1/2, 3/2)
    def curve(L):
        x = t / L ** 1.5
        return L, t, 0.25 + L ** 1.0 * x ** (2 / 3) / (1 + x ** (2 / 3))
    curves = [curve(L) for L in (64, 128, 256)]
    assert A.collapse_spread(curves, 0.5, 1.5) < 1e-2          # ln-ln interpolation on octave-spaced times
    assert A.collapse_spread(curves, 1.0, 1.0) > 0.5          # the Q-TASEP exponents do not collapse KPZ data
    x, y = A.collapse(64, t, curves[0][2], 0.5, 1.5)
    assert np.allclose(y, (t / 512.0) ** (2 / 3) / (1 + (t / 512.0) ** (2 / 3)))


def test_growth_exponent_of_oracle_data_is_in_the_kpz_window():
    L, S = 1024, 24
    times = [2 ** k for k in range(0, 10)]
    sim = R.KpzRef(L, S, 0.75, 0.25, seed=2)
    sim.set_record_times(times)
    sim.run(times[-1])
    r = sim.roughness()
    beta = A.growth_exponent(times, A.w2_mean(L, r["sum_h"], r["sum_h2"]), t_min=16)
    assert 0.25 <= beta <= 0.37, beta


def test_current_fluctuation():
    j_a = np.array([[10, 30], [50, 70]])
    j_b = np.array([[20, 10], [50, 30]])
    mean, c2 = A.current_fluctuation(j_a, j_b, 10)
    assert np.allclose(mean, [0.5, 2.0]) and np.allclose(c2, [(1 + 4) / 2, (0 + 16) / 2])
