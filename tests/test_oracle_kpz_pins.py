"""Pins of the oracle's KPZ/ASEP ring against what the paper and the mathematics fix (no GPU).

Each test names the passage it holds the oracle to.  None of the expected values comes from the oracle
or from the CUDA path: they are closed forms, brute-force master-equation numbers (tests/master_equation.py),
SURVEY.md Appendix B values (tests/golden/), or library routines (numpy cumsum / Fraction arithmetic).
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import master_equation as ME
import workloads
from oracle import kpzref as R

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def flat_words(S, L):
    sites = np.tile(np.arange(L, dtype=np.uint8) & 1, (S, 1))
    return R.pack_sites(sites)


# ------------------------------------------------------------------------------------------------
# Config 1 closed form ("particles would just flip back and forth"; PAPER.md:139 W^2(0)=1/4)
# ------------------------------------------------------------------------------------------------

def test_config1_closed_form_records():
    c = workloads.CONFIGS[1]
    sim = R.KpzRef(c["L"], c["S"], c["p"], c["q"], seed=c["seed"])
    sim.set_record_times(c["record_times"])
    sim.run(c["n_mcs"])
    r = sim.roughness()
    L = c["L"]
    assert list(r["t"]) == c["record_times"]
    assert np.all(r["sum_h2"] == L // 2)
    assert np.all(np.abs(r["sum_h"]) == L // 2)
    assert np.allclose(r["w2_mean"], 0.25, rtol=0, atol=0)
    assert np.all(sim.sites().sum(axis=1) == L // 2)


def test_p1_q0_flat_start_follows_the_offsets():
    # 0101.. -> 1010.. exactly when o=1; 1010.. -> 0101.. exactly when o=0 (SURVEY §8(c) "Config 1 closed form")
    L, S, seed = 64, 6, 1
    sim = R.KpzRef(L, S, 1.0, 0.0, seed=seed)
    sim.set_record_times(list(range(1, 41)))
    zigzag = np.arange(L, dtype=np.uint8) & 1            # 0101..  (Sum h = -L/2)
    state = np.zeros(S, dtype=np.int64)                  # 0 = "0101..", 1 = "1010.."
    for m in range(40):
        sim.run(1)
        for s in range(S):
            for ps in (0, 1):
                o = R.offset(seed, s, m, ps)
                if state[s] == 0 and o == 1:
                    state[s] = 1
                elif state[s] == 1 and o == 0:
                    state[s] = 0
        sites = sim.sites()
        for s in range(S):
            assert np.array_equal(sites[s], zigzag ^ state[s])
    r = sim.roughness()
    # a7: Sum h = -L/2 for 0101.., +L/2 for 1010..; the last record matches the tracked state
    assert np.array_equal(r["sum_h"][-1], np.where(state == 1, L // 2, -L // 2))


def test_alternating_mode_p1_flips_every_mcs_back_to_flat():
    # offset_mode=1 (the paper's even-then-odd order): 0101.. --(o=0: nothing)--> 0101.. --(o=1)--> 1010..;
    # next MCS: o=0 -> 0101.., o=1 -> 1010..  => after every MCS the state is 1010..
    L = 32
    sim = R.KpzRef(L, 2, 1.0, 0.0, seed=3, offset_mode=1)
    for _ in range(5):
        sim.run(1)
        assert np.array_equal(sim.sites()[0], 1 - (np.arange(L) & 1))


# ------------------------------------------------------------------------------------------------
# Trivial parameter cases and invariants
# ------------------------------------------------------------------------------------------------

def test_p0_q0_is_frozen_and_p1_q1_swaps_every_active_pair():
    rng = np.random.default_rng(5)
    L, S, seed = 48, 4, 21
    start = rng.integers(0, 2, size=(S, L), dtype=np.uint8)
    frozen = R.KpzRef(L, S, 0.0, 0.0, seed=seed)
    frozen.set_lattice(R.pack_sites(start))
    frozen.run(7)
    assert np.array_equal(frozen.sites(), start)

    sim = R.KpzRef(L, S, 1.0, 1.0, seed=seed)
    sim.set_lattice(R.pack_sites(start))
    sim.run(5)
    ref = start.copy()
    for m in range(5):
        for s in range(S):
            for ps in (0, 1):
                o = R.offset(seed, s, m, ps)
                a = (2 * np.arange(L // 2) + o) % L
                b = (a + 1) % L
                na, nb = ref[s, a].copy(), ref[s, b].copy()
                ref[s, a], ref[s, b] = nb, na            # every pair (1,0)/(0,1) swaps; (0,0),(1,1) unchanged
    assert np.array_equal(sim.sites(), ref)


@pytest.mark.parametrize("p,q,dis", [(0.75, 0.25, None), (0.9, 0.1, (0.5, 0.3, 0.5, 0.05)), (1.0, 0.0, (0.1, 0.5, 0, 0))])
def test_particle_number_is_conserved(p, q, dis):
    rng = np.random.default_rng(9)
    L, S = 200, 5
    start = (rng.random((S, L)) < 0.37).astype(np.uint8)
    sim = R.KpzRef(L, S, p, q, disorder=dis, seed=8)
    sim.set_lattice(R.pack_sites(start))
    for _ in range(4):
        sim.run(13)
        assert np.array_equal(sim.sites().sum(axis=1), start.sum(axis=1))


def test_sweep_uses_one_uniform_per_pair_departure_site_rates_and_disjoint_pairs():
    """Replay 3 MCS of a ragged ring (150 pairs = 2 supergroups, the second partial) from the per-element
    definition kpzref_uniform/kpzref_offset (32 Philox calls per uniform) — checks the 128-element block
    generation and the pass plumbing against the element-wise definition (Appendix A-5)."""
    rng = np.random.default_rng(11)
    L, seed, sample = 300, 31, 2
    p, q, dis = 0.6, 0.3, (0.4, 0.2, 0.3, 0.9)
    start = (rng.random((1, L)) < 0.5).astype(np.uint8)
    sim = R.KpzRef(L, 1, p, q, disorder=dis, seed=seed, first_sample=sample)
    sim.set_lattice(R.pack_sites(start))
    sp, sq = [R.unpack_words(m, L)[0] for m in sim.disorder_masks()]
    # the masks themselves follow the element-wise definition
    for i in range(0, L, 7):
        assert sp[i] == (R.uniform(seed, R.TAGS["SLOW_P"], sample, 0, 0, i) < R.threshold(dis[0]))
        assert sq[i] == (R.uniform(seed, R.TAGS["SLOW_Q"], sample, 0, 0, i) < R.threshold(dis[2]))
    n = start[0].copy()
    fwd = bwd = 0
    for m in range(3):
        for ps in (0, 1):
            o = R.offset(seed, sample, m, ps)
            for j in range(L // 2):
                a = 2 * j + o
                b = (a + 1) % L
                u = R.uniform(seed, R.TAGS["PAIR"], sample, m, ps, j)
                if n[a] == 1 and n[b] == 0:
                    if u < R.threshold(dis[1] if sp[a] else p):
                        n[a], n[b] = 0, 1
                        fwd += 1
                elif n[a] == 0 and n[b] == 1:
                    if u < R.threshold(dis[3] if sq[b] else q):
                        n[a], n[b] = 1, 0
                        bwd += 1
    sim.run(3)
    assert np.array_equal(sim.sites()[0], n)
    f, b = sim.hops()
    assert (f[0], b[0]) == (fwd, bwd)


def test_resume_and_first_sample_are_exact():
    L, S, seed = 128, 5, 17
    times = [1, 3, 10, 11, 25, 40]
    one = R.KpzRef(L, S, 0.75, 0.25, disorder=(0.2, 0.25, 0.2, 0.75), seed=seed)
    one.set_record_times(times)
    one.run(40)
    two = R.KpzRef(L, S, 0.75, 0.25, disorder=(0.2, 0.25, 0.2, 0.75), seed=seed)
    two.set_record_times(times)
    for n in (7, 4, 0, 19, 10):
        two.run(n)
    assert two.time == 40
    assert np.array_equal(one.lattice(), two.lattice())
    r1, r2 = one.roughness(), two.roughness()
    for k in ("t", "sum_h", "sum_h2"):
        assert np.array_equal(r1[k], r2[k])
    # sample k of an S-sample run == a 1-sample run with first_sample=k (RNG keyed by global sample index)
    k = 3
    solo = R.KpzRef(L, 1, 0.75, 0.25, disorder=(0.2, 0.25, 0.2, 0.75), seed=seed, first_sample=k)
    solo.set_record_times(times)
    solo.run(40)
    assert np.array_equal(solo.lattice()[0], one.lattice()[k])
    assert np.array_equal(solo.roughness()["sum_h2"][:, 0], r1["sum_h2"][:, k])
    assert np.array_equal(solo.disorder_masks()[0][0], one.disorder_masks()[0][k])


def test_disorder_mask_density():
    # Eq. 8: a site is slow with probability Q, independently
    L, S = 4096, 4
    sim = R.KpzRef(L, S, 1.0, 0.0, disorder=(0.1, 0.5, 0.35, 0.0), seed=3)
    sp, sq = [R.unpack_words(m, L) for m in sim.disorder_masks()]
    n = L * S
    assert abs(sp.mean() - 0.1) < 5 * np.sqrt(0.1 * 0.9 / n)
    assert abs(sq.mean() - 0.35) < 5 * np.sqrt(0.35 * 0.65 / n)
    assert abs(np.corrcoef(sp.ravel(), sq.ravel())[0, 1]) < 5 / np.sqrt(n)   # independent masks (§R8)
    assert not np.array_equal(sp[0], sp[1])                                  # per-sample realisations


# ------------------------------------------------------------------------------------------------
# Heights and width (PAPER.md:105-108 Eq. 3, :139)
# ------------------------------------------------------------------------------------------------

def test_flat_state_width_is_one_quarter():
    for L in (4, 64, 1000):
        sim = R.KpzRef(L, 1, 0.5, 0.5, seed=1)
        sim.set_record_times([1])
        h = sim.heights(0)
        assert np.array_equal(h, np.where(np.arange(L) % 2 == 0, -1, 0))
        assert Fraction(int((h.astype(np.int64) ** 2).sum()), L) - Fraction(int(h.sum()), L) ** 2 == Fraction(1, 4)


def test_tent_profile_closed_form_sums():
    # n = 1^k 0^(L-k): h_x = x+1 for x<k, then k-(x+1-k) = 2k-x-1 for x>=k.  Closed-form power sums.
    L, k = 90, 37
    sites = np.zeros((1, L), dtype=np.uint8)
    sites[0, :k] = 1
    sim = R.KpzRef(L, 1, 0.0, 0.0, seed=1)
    sim.set_lattice(R.pack_sites(sites))
    sim.set_record_times([1])
    sim.run(1)                                   # p=q=0: frozen, the record is of the tent itself
    r = sim.roughness()

    def s1(n):
        return n * (n + 1) // 2

    def s2(n):
        return n * (n + 1) * (2 * n + 1) // 6
    # rising part: 1..k ; falling part: values k-1, k-2, ..., k-(L-k) = 2k-L
    lo = 2 * k - L
    fall1 = (s1(k - 1) - s1(lo - 1)) if lo >= 1 else (s1(k - 1) - s1(-lo))          # sum of lo..k-1
    fall2 = (s2(k - 1) - s2(lo - 1)) if lo >= 1 else (s2(k - 1) + s2(-lo))          # sum of squares lo..k-1
    assert r["sum_h"][0, 0] == s1(k) + fall1
    assert r["sum_h2"][0, 0] == s2(k) + fall2
    assert sim.heights(0)[-1] == 2 * k - L       # h_{L-1} = 2N - L


def test_heights_match_library_prefix_sum_and_w2_mean_matches_exact_fractions():
    rng = np.random.default_rng(2)
    L, S = 77 * 2, 6
    sites = (rng.random((S, L)) < 0.45).astype(np.uint8)
    sim = R.KpzRef(L, S, 0.0, 0.0, seed=4)
    sim.set_lattice(R.pack_sites(sites))
    sim.set_record_times([2])
    sim.run(2)
    r = sim.roughness()
    w2 = Fraction(0)
    for s in range(S):
        h = np.cumsum(2 * sites[s].astype(np.int64) - 1)
        assert np.array_equal(sim.heights(s), h)
        assert h[-1] == 2 * int(sites[s].sum()) - L
        assert r["sum_h"][0, s] == h.sum() and r["sum_h2"][0, s] == (h * h).sum()
        w2 += Fraction(int((h * h).sum()), L) - Fraction(int(h.sum()), L) ** 2
    assert r["w2_mean"][0] == pytest.approx(float(w2 / S), rel=1e-14)


# ------------------------------------------------------------------------------------------------
# Master equation (acceptance rule, rate site, schedule): SURVEY §8(c), Appendix B-3
# ------------------------------------------------------------------------------------------------

def _golden_currents():
    rows = []
    with open(os.path.join(GOLDEN, "master_equation_currents.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            v = line.split()
            rows.append(dict(L=int(v[0]), N=int(v[1]), p=float(v[2]), q=float(v[3]), slow=int(v[4]),
                             p_slow=float(v[5]), alternating=float(v[6]), drawn=float(v[7]), rsu=float(v[8])))
    return rows


def _rates(row):
    ps = [row["p"]] * row["L"]
    if row["slow"] >= 0:
        ps[row["slow"]] = row["p_slow"]
    return ps, [row["q"]] * row["L"]


def test_brute_force_master_equation_reproduces_survey_currents():
    for row in _golden_currents():
        ps, qs = _rates(row)
        for mode in ("alternating", "drawn"):
            assert ME.kpz_current_per_bond(row["L"], row["N"], ps, qs, mode) == pytest.approx(row[mode], abs=2e-12)
        if row["slow"] < 0:
            L, N = row["L"], row["N"]
            assert (row["p"] - row["q"]) * N * (L - N) / (L * (L - 1)) == pytest.approx(row["rsu"], abs=1e-12)


def _oracle_current(row, mode, S, burn, n_mcs, seed):
    L, N = row["L"], row["N"]
    dis = None
    if row["slow"] >= 0:
        dis = (0.0, row["p_slow"], 0.0, 0.0)
    sim = R.KpzRef(L, S, row["p"], row["q"], disorder=dis, seed=seed, offset_mode=1 if mode == "alternating" else 0)
    sites = np.zeros((S, L), dtype=np.uint8)
    sites[:, :2 * N:2] = 1                        # N particles on even sites 0,2,..: any start works (stationary)
    sim.set_lattice(R.pack_sites(sites))
    if row["slow"] >= 0:
        mask = np.zeros((S, L), dtype=np.uint8)
        mask[:, row["slow"]] = 1
        sim.set_disorder_masks(slow_p=R.pack_sites(mask))
    if mode == "rsu":
        sim.run_rsu(burn)
    else:
        sim.run(burn)
    f0, b0 = sim.hops()
    if mode == "rsu":
        sim.run_rsu(n_mcs)
    else:
        sim.run(n_mcs)
    f1, b1 = sim.hops()
    j = ((f1 - f0) - (b1 - b0)) / float(L * n_mcs)
    return j.mean(), j.std(ddof=1) / np.sqrt(S)


@pytest.mark.parametrize("idx,mode", [(1, "drawn"), (1, "alternating"), (3, "drawn"), (2, "drawn"),
                                      (7, "drawn"), (7, "alternating"), (1, "rsu"), (3, "rsu"),
                                      (6, "drawn"), (6, "alternating"), (6, "rsu")])  # row 6: p=0.9, q=0.1 (32 planes)
def test_oracle_stationary_current_matches_master_equation(idx, mode):
    row = _golden_currents()[idx]
    if mode == "alternating" and row["slow"] >= 0:
        # p=1 away from the slow site under strict alternation: stationary current 1/2 (golden line)
        pass
    mean, sem = _oracle_current(row, mode, S=192, burn=200, n_mcs=3000, seed=1000 + idx)
    exact = row[mode]
    assert abs(mean - exact) < 5 * sem + 1e-12, (mean, exact, sem)
    # resolution: the three schedules differ by >= 7 %; the measurement resolves 1.5 %
    assert 5 * sem < 0.015 * exact + 1e-12


def test_finite_time_distribution_with_slow_sites_chi2():
    """Exact distribution after 2 MCS from the flat state with one slow-p and one slow-q site versus the oracle's
    histogram over 40000 samples.  The alternative readings (rate indexed by the arrival site; p and q swapped)
    are shown to be rejected by the same data, so the test has the power to catch them."""
    L, N, S, t = 8, 4, 40000, 2
    p, q, p_slow, q_slow = 0.75, 0.25, 0.25, 0.75
    sp_site, sq_site = 3, 6
    flat = sum(1 << i for i in range(1, L, 2))                   # n_i = i & 1
    ps = [p] * L
    qs = [q] * L
    ps[sp_site] = p_slow
    qs[sq_site] = q_slow
    states, v, fwd, bwd = ME.kpz_finite_time(L, N, ps, qs, flat, t, "drawn")

    sim = R.KpzRef(L, S, p, q, disorder=(0.0, p_slow, 0.0, q_slow), seed=77)
    mp = np.zeros((S, L), dtype=np.uint8)
    mq = np.zeros((S, L), dtype=np.uint8)
    mp[:, sp_site] = 1
    mq[:, sq_site] = 1
    sim.set_disorder_masks(R.pack_sites(mp), R.pack_sites(mq))
    sim.run(t)
    codes = sim.lattice()[:, 0].astype(np.int64)
    counts = np.array([(codes == s).sum() for s in states], dtype=np.float64)
    assert counts.sum() == S

    def chi2(prob):
        keep = prob * S >= 5
        rest_obs, rest_exp = counts[~keep].sum(), prob[~keep].sum() * S
        c = ((counts[keep] - prob[keep] * S) ** 2 / (prob[keep] * S)).sum()
        if rest_exp > 0:
            c += (rest_obs - rest_exp) ** 2 / rest_exp
        return c, int(keep.sum())

    c, dof = chi2(v)
    assert c < dof + 5 * np.sqrt(2 * dof), (c, dof)
    # expected accepted moves (PAPER.md:95 rates) — also exact
    f, b = sim.hops()
    assert abs(f.mean() - fwd) < 5 * f.std(ddof=1) / np.sqrt(S)
    assert abs(b.mean() - bwd) < 5 * b.std(ddof=1) / np.sqrt(S)
    # alternative readings are rejected by the same histogram
    ps_arrival = [p] * L
    ps_arrival[(sp_site - 1) % L] = p_slow                       # "p of the arrival site"
    qs_arrival = [q] * L
    qs_arrival[(sq_site + 1) % L] = q_slow
    _, v_alt, _, _ = ME.kpz_finite_time(L, N, ps_arrival, qs_arrival, flat, t, "drawn")
    assert chi2(v_alt)[0] > 20 * dof
    _, v_alt2, _, _ = ME.kpz_finite_time(L, N, ps, qs, flat, t, "alternating")
    assert chi2(v_alt2)[0] > 20 * dof
    _, v_swapped, _, _ = ME.kpz_finite_time(L, N, qs, ps, flat, t, "drawn")
    assert chi2(v_swapped)[0] > 20 * dof


@pytest.mark.parametrize("p,q,p_slow,q_slow", [(0.3, 0.6, 0.9, 0.1), (0.9, 0.1, 0.8, 1.0 / 3.0)])
def test_finite_time_distribution_non_dyadic_rates_chi2(p, q, p_slow, q_slow):
    """As above with rates whose thresholds use all 32 bit-planes (0.3 -> 0x4CCCCCCC, 0.6 -> 0x99999999, 0.9, 0.1, 0.8,
    1/3): the acceptance comparison has to be right beyond the two leading planes.  Power: the
    same histogram rejects the distribution for rates rounded to their 2 leading bits."""
    L, N, S, t = 8, 4, 60000, 2
    sp_site, sq_site = 2, 5
    flat = sum(1 << i for i in range(1, L, 2))
    ps, qs = [p] * L, [q] * L
    ps[sp_site], qs[sq_site] = p_slow, q_slow
    states, v, fwd, bwd = ME.kpz_finite_time(L, N, ps, qs, flat, t, "drawn")
    sim = R.KpzRef(L, S, p, q, disorder=(0.0, p_slow, 0.0, q_slow), seed=78)
    mp = np.zeros((S, L), dtype=np.uint8)
    mq = np.zeros((S, L), dtype=np.uint8)
    mp[:, sp_site] = 1
    mq[:, sq_site] = 1
    sim.set_disorder_masks(R.pack_sites(mp), R.pack_sites(mq))
    sim.run(t)
    codes = sim.lattice()[:, 0].astype(np.int64)
    counts = np.array([(codes == s).sum() for s in states], dtype=np.float64)
    assert counts.sum() == S

    def chi2(prob):
        keep = prob * S >= 5
        c = ((counts[keep] - prob[keep] * S) ** 2 / (prob[keep] * S)).sum()
        rest_exp = prob[~keep].sum() * S
        if rest_exp > 0:
            c += (counts[~keep].sum() - rest_exp) ** 2 / rest_exp
        return c, int(keep.sum())

    c, dof = chi2(v)
    assert c < dof + 5 * np.sqrt(2 * dof), (c, dof)
    f, b = sim.hops()
    assert abs(f.mean() - fwd) < 5 * f.std(ddof=1) / np.sqrt(S)
    assert abs(b.mean() - bwd) < 5 * b.std(ddof=1) / np.sqrt(S)
    trunc = lambda x: np.floor(x * 4) / 4                        # what a comparison of the 2 leading planes would give
    _, v2, _, _ = ME.kpz_finite_time(L, N, [trunc(x) for x in ps], [trunc(x) for x in qs], flat, t, "drawn")
    assert chi2(v2)[0] > 20 * dof
    trunc4 = lambda x: np.floor(x * 16) / 16                     # ... of the 4 leading planes
    _, v4, _, _ = ME.kpz_finite_time(L, N, [trunc4(x) for x in ps], [trunc4(x) for x in qs], flat, t, "drawn")
    assert chi2(v4)[0] > dof + 8 * np.sqrt(2 * dof)


def test_stationary_width_matches_master_equation():
    # Appendix B-3: stationary E[W^2] after a full MCS, L=8 p=.75 q=.25: 0.700338600451 (drawn);
    # re-derived here by brute force, then measured on the oracle.
    L, N, p, q = 8, 4, 0.75, 0.25
    states = ME.sector_states(L, N)
    T0, _, _ = ME.kpz_pass(L, states, 0, [p] * L, [q] * L)
    T1, _, _ = ME.kpz_pass(L, states, 1, [p] * L, [q] * L)
    pi = ME.stationary(0.5 * (T0 + T1))
    exact = float(sum(pr * ME.width2(s, L) for s, pr in zip(states, pi)))
    assert exact == pytest.approx(0.700338600451, abs=1e-11)
    S, burn, n = 128, 100, 1500
    sim = R.KpzRef(L, S, p, q, seed=5)
    sim.set_record_times(list(range(burn + 1, burn + n + 1)))
    sim.run(burn + n)
    r = sim.roughness()
    w2 = (L * r["sum_h2"] - r["sum_h"] ** 2) / float(L * L)            # [n][S]
    per_sample = w2.mean(axis=0)
    assert abs(per_sample.mean() - exact) < 5 * per_sample.std(ddof=1) / np.sqrt(S)
    assert r["w2_mean"] == pytest.approx(w2.mean(axis=1), rel=1e-13)


# ------------------------------------------------------------------------------------------------
# Random-sequential mode closed forms (north_star "J = p N (L-N) / (L (L-1))")
# ------------------------------------------------------------------------------------------------

def test_rsu_half_filled_stationary_width_is_L_plus_1_over_12():
    # uniform stationary measure of the exclusion process on a ring at half filling: E[W^2] = (L+1)/12 (Appendix B-4)
    L, S, burn, n = 16, 96, 300, 1200
    states = ME.sector_states(L, L // 2)
    assert np.mean([ME.width2(s, L) for s in states]) == pytest.approx((L + 1) / 12.0, abs=1e-12)
    sim = R.KpzRef(L, S, 0.7, 0.2, seed=12)
    sim.set_record_times(list(range(burn + 1, burn + n + 1, 3)))
    sim.run_rsu(burn + n)
    r = sim.roughness()
    w2 = (L * r["sum_h2"] - r["sum_h"] ** 2) / float(L * L)
    per_sample = w2.mean(axis=0)
    assert abs(per_sample.mean() - (L + 1) / 12.0) < 5 * per_sample.std(ddof=1) / np.sqrt(S)
    assert 5 * per_sample.std(ddof=1) / np.sqrt(S) < 0.03 * (L + 1) / 12.0


def test_rsu_tasep_current_closed_form():
    L, N, S, p = 20, 7, 128, 0.8
    sim = R.KpzRef(L, S, p, 0.0, seed=13)
    sites = np.zeros((S, L), dtype=np.uint8)
    sites[:, :N] = 1
    sim.set_lattice(R.pack_sites(sites))
    sim.run_rsu(300)
    f0, _ = sim.hops()
    n = 2500
    sim.run_rsu(n)
    f1, b1 = sim.hops()
    assert np.all(b1 == 0)
    j = (f1 - f0) / float(L * n)
    exact = R.threshold(p) / 2.0**32 * N * (L - N) / (L * (L - 1))
    assert abs(j.mean() - exact) < 5 * j.std(ddof=1) / np.sqrt(S)
    assert 5 * j.std(ddof=1) / np.sqrt(S) < 0.01 * exact


# ------------------------------------------------------------------------------------------------
# KPZ growth (PAPER.md:112 Eq. 4, :139 alpha=1/2, z=3/2 => beta=1/3)
# ------------------------------------------------------------------------------------------------

def test_kpz_growth_exponent_window():
    L, S = 2048, 40
    times = [2 ** k for k in range(0, 11)]
    sim = R.KpzRef(L, S, 0.75, 0.25, seed=2)
    sim.set_record_times(times)
    sim.run(times[-1])
    r = sim.roughness()
    w2 = r["w2_mean"] - 0.25                      # subtract the intrinsic width of the zig-zag
    t = np.array(times, dtype=np.float64)
    sel = t >= 32
    slope = np.polyfit(np.log(t[sel]), np.log(w2[sel]), 1)[0]
    beta = 0.5 * slope
    assert 0.26 <= beta <= 0.36, beta
    assert np.all(np.diff(w2) > 0)                # roughening, no saturation yet (t << L^{3/2})


def test_set_time_restores_a_checkpoint_exactly():
    """lattice + t (+ quenched tags, regenerated from the seed) are the whole state."""
    L, S, a, b = 192, 3, 23, 31
    full = R.KpzRef(L, S, 0.8, 0.1, disorder=(0.3, 0.2, 0.3, 0.05), seed=61)
    full.set_record_times([a + b])
    full.run(a + b)
    part = R.KpzRef(L, S, 0.8, 0.1, disorder=(0.3, 0.2, 0.3, 0.05), seed=61)
    part.run(a)
    fresh = R.KpzRef(L, S, 0.8, 0.1, disorder=(0.3, 0.2, 0.3, 0.05), seed=61)
    fresh.set_lattice(part.lattice())
    fresh.set_time(a)
    fresh.set_record_times([a + b])
    fresh.run(b)
    assert fresh.time == a + b
    assert np.array_equal(fresh.lattice(), full.lattice())
    assert np.array_equal(fresh.roughness()["sum_h2"], full.roughness()["sum_h2"])
    with pytest.raises(R.OracleError):
        fresh.set_time(-1)
    with pytest.raises(R.OracleError):
        fresh.set_time(1 << 54)
