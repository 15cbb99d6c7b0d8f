"""Pins of the oracle's two-lane model — no GPU.

Expected values: brute-force two-lane master equation on L=4 (tests/master_equation.py), conservation laws,
the left/right symmetry the paper states, and the oracle's own KPZ ring (already pinned by
tests/test_oracle_kpz_pins.py) for the omega=0 reduction.
"""
import numpy as np
import pytest

import master_equation as ME
from oracle import kpzref as R


def test_total_particle_number_is_conserved_and_per_lane_when_no_turning_points():
    L, S = 256, 6
    sim = R.LanesRef(L, S, 1.0, 1.0, 0.3, 0.05, 10, 0.1, seed=5)
    n0 = sim.totals()
    for _ in range(5):
        sim.run(17)
        n = sim.totals()
        assert np.array_equal(n["n_a"] + n["n_b"], n0["n_a"] + n0["n_b"])
    assert not np.array_equal(n["n_a"], n0["n_a"])           # lanes do exchange particles
    iso = R.LanesRef(L, S, 0.5, 0.5, 0.3, 0.0, 10, 0.9, seed=5)
    m0 = iso.totals()
    iso.run(60)
    m = iso.totals()
    assert np.array_equal(m["n_a"], m0["n_a"]) and np.array_equal(m["n_b"], m0["n_b"])


def test_initial_and_turning_point_densities_and_epoch_redraw():
    L, S, seed, period = 2048, 4, 5, 7
    sim = R.LanesRef(L, S, 1.0, 1.0, 0.3, 0.05, period, 0.1, seed=seed)
    a, b, turn = [R.unpack_words(x, L) for x in sim.state()]
    n = L * S
    assert abs(a.mean() - 0.3) < 5 * np.sqrt(0.21 / n)
    assert abs(b.mean() - 0.3) < 5 * np.sqrt(0.21 / n)
    assert abs(turn.mean() - 0.05) < 5 * np.sqrt(0.05 * 0.95 / n)
    assert abs(np.corrcoef(a.ravel(), b.ravel())[0, 1]) < 5 / np.sqrt(n)
    # element-wise definition of the streams (§R14)
    for i in range(0, L, 97):
        assert a[1, i] == (R.uniform(seed, R.TAGS["INIT_A"], 1, 0, 0, i) < R.threshold(0.3))
        assert b[1, i] == (R.uniform(seed, R.TAGS["INIT_B"], 1, 0, 0, i) < R.threshold(0.3))
        assert turn[1, i] == (R.uniform(seed, R.TAGS["TURN"], 1, 0, 0, i) < R.threshold(0.05))
    sim.run(period)                     # MCS 0..period-1 use epoch 0: mask unchanged
    assert np.array_equal(R.unpack_words(sim.state()[2], L), turn)
    sim.run(1)                          # MCS index `period` starts epoch 1
    turn1 = R.unpack_words(sim.state()[2], L)
    assert not np.array_equal(turn1, turn)
    for i in range(0, L, 97):
        assert turn1[2, i] == (R.uniform(seed, R.TAGS["TURN"], 2, 1, 0, i) < R.threshold(0.05))
    never = R.LanesRef(L, 1, 1.0, 1.0, 0.3, 0.05, 0, 0.1, seed=seed)
    t0 = never.state()[2].copy()
    never.run(30)
    assert np.array_equal(never.state()[2], t0)


def test_lane_a_reduces_to_the_kpz_ring_when_lanes_are_decoupled():
    # omega = 0: lane A is a TASEP ring with the PAIR and OFFSET streams of the KPZ sweep (Appendix A-2)
    L, S, seed, p_a = 192, 3, 19, 0.75
    lanes = R.LanesRef(L, S, p_a, 0.5, 0.3, 0.05, 10, 0.0, seed=seed)
    a0, b0, _ = lanes.state()
    ring = R.KpzRef(L, S, p_a, 0.0, seed=seed)
    ring.set_lattice(a0)
    lanes.run(25)
    ring.run(25)
    assert np.array_equal(lanes.state()[0], ring.lattice())
    assert np.array_equal(lanes.totals()["j_a"], ring.hops()[0])
    # lane B moved (to the left): its particle number is unchanged, its configuration is not
    assert not np.array_equal(lanes.state()[1], b0)


def test_lane_b_hops_left_lane_a_hops_right():
    L = 16
    sim = R.LanesRef(L, 1, 1.0, 1.0, 0.0, 0.0, 0, 0.0, seed=3)
    a = np.zeros((1, L), dtype=np.uint8)
    b = np.zeros((1, L), dtype=np.uint8)
    a[0, 5] = 1
    b[0, 5] = 1
    sim.set_state(R.pack_sites(a), R.pack_sites(b))
    sim.run(1)
    A, B, _ = [R.unpack_words(x, L)[0] for x in sim.state()]
    tot = sim.totals()
    # a single particle with rate 1 hops once per pass in which its bond is active: displacement = hops
    assert A.sum() == 1 and B.sum() == 1
    assert np.argmax(A) == (5 + tot["j_a"][0]) % L
    assert np.argmax(B) == (5 - tot["j_b"][0]) % L
    # over many MCS both move, in opposite directions
    sim.run(40)
    tot = sim.totals()
    assert tot["j_a"][0] > 10 and tot["j_b"][0] > 10


@pytest.mark.parametrize("p_a,p_b,omega,turn_mask,start", [
    (0.5, 0.5, 0.8, 0b0101, (0b0011, 0b0100)),
    (1.0, 1.0, 0.1, 0b0010, (0b1001, 0b0001)),
    (0.75, 0.25, 0.5, 0b1111, (0b0001, 0b0110)),
    (0.3, 0.6, 0.1, 0b1111, (0b0101, 0b0010)),      # every threshold uses all 32 bit-planes (omega = 0.1 as in config 5)
])
def test_finite_time_two_lane_master_equation(p_a, p_b, omega, turn_mask, start):
    """Exact distribution and expected hop counts after 3 MCS on L=4 versus the oracle's histogram over 30000
    samples.  Pins the 4-step order (in-lane, A->B, in-lane, B->A), the hop directions, the
    switch rule (source occupied, target empty, turning point) and the shared offset (§R12)."""
    L, S, t = 4, 30000, 3
    A0, B0 = start
    states, v, JA, JB = ME.lanes_finite_time(L, A0 | (B0 << L), turn_mask, p_a, p_b, omega, t)
    sim = R.LanesRef(L, S, p_a, p_b, 0.5, 0.5, 0, omega, seed=101)
    ones = np.ones((S, 1), dtype=np.uint32)
    sim.set_state(ones * A0, ones * B0, ones * turn_mask)
    sim.run(t)
    a, b, _ = sim.state()
    codes = a[:, 0].astype(np.int64) | (b[:, 0].astype(np.int64) << L)
    counts = np.array([(codes == s).sum() for s in states], dtype=np.float64)
    assert counts.sum() == S
    keep = v * S >= 5
    chi2 = ((counts[keep] - v[keep] * S) ** 2 / (v[keep] * S)).sum()
    if v[~keep].sum() > 0:
        chi2 += (counts[~keep].sum() - v[~keep].sum() * S) ** 2 / (v[~keep].sum() * S)
    dof = int(keep.sum())
    assert chi2 < dof + 5 * np.sqrt(2 * dof), (chi2, dof)
    assert counts[v == 0].sum() == 0                      # nothing lands on an unreachable state
    tot = sim.totals()
    for got, exact in ((tot["j_a"], JA), (tot["j_b"], JB)):
        sem = got.std(ddof=1) / np.sqrt(S)
        assert abs(got.mean() - exact) < 5 * sem + 1e-12
        assert 5 * sem < 0.05 * max(exact, 0.2)
    # power: swapping the order of the two lane-change steps is rejected by the same histogram
    _, v_alt, _, _ = ME.lanes_finite_time(L, A0 | (B0 << L), turn_mask, p_a, p_b, omega, t, ab_first=False)
    ok = v_alt * S >= 5
    chi2_alt = ((counts[ok] - v_alt[ok] * S) ** 2 / (v_alt[ok] * S)).sum()
    assert chi2_alt > 10 * dof, (chi2_alt, dof)


def test_currents_are_symmetric_at_equal_densities():
    # PAPER.md:253 "the total current of particles vanishes due to the left/right symmetry"
    L, S = 128, 64
    sim = R.LanesRef(L, S, 1.0, 1.0, 0.3, 0.05, 100, 0.1, seed=5)
    sim.set_record_times([50, 400])
    sim.run(400)
    c = sim.currents()
    net = (c["j_a"][1] - c["j_a"][0]) - (c["j_b"][1] - c["j_b"][0])
    assert abs(net.mean()) < 5 * net.std(ddof=1) / np.sqrt(S)
    assert c["j_a"][1].mean() > 1000        # both lanes carry current
    assert np.array_equal(c["n_a"][1] + c["n_b"][1], c["n_a"][0] + c["n_b"][0])


def test_profile_accumulates_at_epoch_ends():
    L, S, period = 64, 2, 5
    sim = R.LanesRef(L, S, 0.0, 0.0, 0.4, 0.3, period, 0.0, seed=8)       # frozen dynamics
    a0, b0, _ = [R.unpack_words(x, L) for x in sim.state()]
    sim.run(period - 1)
    assert sim.profile()[2] == 0
    sim.run(1)
    assert sim.profile()[2] == 1
    sim.run(3 * period + 2)
    oa, ob, ns = sim.profile()
    assert ns == 4
    assert np.array_equal(oa, 4 * a0.astype(np.uint32)) and np.array_equal(ob, 4 * b0.astype(np.uint32))


def test_lanes_resume_and_first_sample_are_exact():
    L, S, seed = 128, 4, 23
    times = [2, 9, 10, 31]
    args = (0.75, 0.5, 0.3, 0.2, 10, 0.3)
    one = R.LanesRef(L, S, *args, seed=seed)
    one.set_record_times(times)
    one.run(31)
    two = R.LanesRef(L, S, *args, seed=seed)
    two.set_record_times(times)
    for n in (10, 1, 9, 11):
        two.run(n)
    for x, y in zip(one.state(), two.state()):
        assert np.array_equal(x, y)
    c1, c2 = one.currents(), two.currents()
    for k in c1:
        assert np.array_equal(c1[k], c2[k])
    assert np.array_equal(one.profile()[0], two.profile()[0]) and one.profile()[2] == two.profile()[2] == 3
    solo = R.LanesRef(L, 1, *args, seed=seed, first_sample=2)
    solo.set_record_times(times)
    solo.run(31)
    assert np.array_equal(solo.state()[0][0], one.state()[0][2])
    assert np.array_equal(solo.currents()["j_b"][:, 0], c1["j_b"][:, 2])


# ---------------------------------------------------------------------------------------------------------
# the paper's own two-lane model - every site can be crossed, with probability
# omega where its flag is set and w_unflagged elsewhere; separate flag sets u_i (A->B) and v_i (B->A)
# ---------------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("p_a,p_b,w1,w0,mask_u,mask_v,start", [
    (0.5, 0.5, 0.2, 0.8, 0b0101, 0b0011, (0b0011, 0b0100)),     # the paper's rates
    (1.0, 0.75, 0.5, 0.25, 0b1000, 0b0110, (0b1001, 0b0010)),
])
def test_crossing_model_finite_time_master_equation(p_a, p_b, w1, w0, mask_u, mask_v, start):
    """Exact distribution after 3 MCS on L=4 versus 30000 oracle samples: pins that unflagged sites cross with
    w_unflagged, flagged ones with omega, and that A->B reads the flags u while B->A reads v."""
    L, S, t = 4, 30000, 3
    A0, B0 = start
    states, v, JA, JB = ME.lanes_finite_time(L, A0 | (B0 << L), mask_u, p_a, p_b, w1, t, w_unflagged=w0, mask_v=mask_v)
    sim = R.LanesRef(L, S, p_a, p_b, 0.5, 0.5, 0, w1, seed=202, w_unflagged=w0, independent=1)
    ones = np.ones((S, 1), dtype=np.uint32)
    sim.set_state(ones * A0, ones * B0)
    sim.set_flags(ones * mask_u, ones * mask_v)
    sim.run(t)
    a, b, _ = sim.state()
    codes = a[:, 0].astype(np.int64) | (b[:, 0].astype(np.int64) << L)
    counts = np.array([(codes == s).sum() for s in states], dtype=np.float64)
    keep = v * S >= 5
    chi2 = ((counts[keep] - v[keep] * S) ** 2 / (v[keep] * S)).sum()
    if v[~keep].sum() > 0:
        chi2 += (counts[~keep].sum() - v[~keep].sum() * S) ** 2 / (v[~keep].sum() * S)
    dof = int(keep.sum())
    assert chi2 < dof + 5 * np.sqrt(2 * dof), (chi2, dof)
    tot = sim.totals()
    for got, exact in ((tot["j_a"], JA), (tot["j_b"], JB)):
        assert abs(got.mean() - exact) < 5 * got.std(ddof=1) / np.sqrt(S) + 1e-12
    # power: swapping the roles of u and v, or of the two crossing probabilities, is rejected
    for alt in (dict(turn_mask=mask_v, mask_v=mask_u, omega=w1, w_unflagged=w0),
                dict(turn_mask=mask_u, mask_v=mask_v, omega=w0, w_unflagged=w1)):
        _, v_alt, _, _ = ME.lanes_finite_time(L, A0 | (B0 << L), alt["turn_mask"], p_a, p_b, alt["omega"], t,
                                              w_unflagged=alt["w_unflagged"], mask_v=alt["mask_v"])
        ok = v_alt * S >= 5
        chi2_alt = ((counts[ok] - v_alt[ok] * S) ** 2 / (v_alt[ok] * S)).sum()
        assert chi2_alt > 10 * dof, (chi2_alt, dof)


def test_crossing_model_flags_conservation_and_reduction_to_the_turning_point_model():
    L, S, seed = 512, 4, 77
    sim = R.LanesRef(L, S, 0.5, 0.5, 0.5, 0.5, 0, 0.2, seed=seed, w_unflagged=0.8, independent=1)
    u, v = [R.unpack_words(x, L) for x in sim.flags()]
    assert not np.array_equal(u, v)
    n = S * L
    for f in (u, v):
        assert abs(f.mean() - 0.5) < 5 * np.sqrt(0.25 / n)
    for i in (0, 1, 129, L - 1):       # u from stream TURN, v from stream TURN_V, epoch 0
        assert u[1, i] == (R.uniform(seed, R.TAGS["TURN"], 1, 0, 0, i) < R.threshold(0.5))
        assert v[1, i] == (R.uniform(seed, R.TAGS["TURN_V"], 1, 0, 0, i) < R.threshold(0.5))
    a0, b0, _ = sim.state()
    n0 = R.unpack_words(a0, L).sum(axis=1) + R.unpack_words(b0, L).sum(axis=1)
    sim.run(50)
    a1, b1, _ = sim.state()
    assert np.array_equal(R.unpack_words(a1, L).sum(axis=1) + R.unpack_words(b1, L).sum(axis=1), n0)
    assert np.array_equal(R.unpack_words(sim.flags()[0], L), u)        # quenched: period 0
    # w_unflagged = 0 with one shared flag set IS the turning-point model, bit for bit
    x = R.LanesRef(L, S, 1.0, 1.0, 0.3, 0.05, 7, 0.1, seed=5)
    y = R.LanesRef(L, S, 1.0, 1.0, 0.3, 0.05, 7, 0.1, seed=5, w_unflagged=0.0, independent=0)
    x.run(30)
    y.run(30)
    for p, q in zip(x.state(), y.state()):
        assert np.array_equal(p, q)
    with pytest.raises(R.OracleError):
        y.set_flags(None, np.zeros((S, L // 32), dtype=np.uint32))      # one shared set: there is no separate v
