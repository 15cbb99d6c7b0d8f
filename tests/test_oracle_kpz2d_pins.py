"""Pins of the 2+1D oracle (oracle/kpz2d_oracle.c; "checker-board lattice decomposition in two
dimensions") - no GPU.  The model is this repository's reading of a one-sentence outlook; what is pinned is
that the oracle implements that reading: closed form, invariants of a single-valued height field, a brute-force master
equation on a 4 x 4 lattice that rejects the plausible wrong readings, the particle-hole symmetry, resume."""
import numpy as np
import pytest

import master_equation as ME
from oracle import kpzref as R


def _bits(words, Lx):
    """[S][Ly][words] uint32 -> [S][Ly][Lx] uint8."""
    x = np.arange(Lx)
    return ((words[..., x >> 5] >> (x & 31).astype(np.uint32)) & 1).astype(np.uint8)


def test_flat_start_has_width_one_quarter_and_the_documented_slopes():
    Lx, Ly = 8, 6
    sim = R.Kpz2dRef(Lx, Ly, 2, 0.5, 0.5, seed=1)
    sx, sy = sim.slopes()
    want = np.array([[(x + y) & 1 for x in range(Lx)] for y in range(Ly)], dtype=np.uint8)
    assert np.array_equal(_bits(sx, Lx)[0], want) and np.array_equal(_bits(sy, Lx)[1], want)
    h = sim.heights(0)
    assert np.array_equal(h, want.astype(np.int32) - 1)            # h(0,0) = 2 sx[0][0] - 1 = -1 (DESIGN §R5 carried over)
    N = Lx * Ly
    assert (N * (h.astype(np.int64) ** 2).sum() - h.sum() ** 2) / N ** 2 == 0.25


def test_p_one_q_zero_flips_between_the_two_flat_surfaces_exactly_when_the_colour_matches():
    """The 2+1D analogue of config 1 ("particles would just flip back and forth"): from the flat start with
    p = 1, q = 0 all local maxima - the sites of one colour - move together exactly when the pass draws their colour."""
    Lx, Ly, S, T, seed = 8, 4, 5, 40, 11
    sim = R.Kpz2dRef(Lx, Ly, S, 1.0, 0.0, seed=seed)
    sim.set_record_times(list(range(1, T + 1)))
    sim.run(T)
    r = sim.roughness()
    N = Lx * Ly
    for s in range(S):
        mu = 1                                                       # colour of the maxima: (x + y) & 1 == mu
        for m in range(T):
            for ps in range(2):
                if R.offset(seed, s, m, ps) == mu:
                    mu ^= 1
            assert r["sum_h"][m, s] == (-N // 2 if mu == 1 else N // 2), (s, m)
            assert r["sum_h2"][m, s] == N // 2
    assert np.all(r["w2_mean"] == 0.25)
    f, b = sim.hops()
    assert np.all(b == 0) and np.all(f % (N // 2) == 0)


@pytest.mark.parametrize("p,q,mode", [(0.75, 0.25, 0), (0.9, 0.1, 1), (0.3, 0.6, 0)])
def test_height_field_stays_single_valued(p, q, mode):
    Lx, Ly, S = 16, 10, 3
    sim = R.Kpz2dRef(Lx, Ly, S, p, q, seed=5, offset_mode=mode)
    sim.run(60)
    sx, sy = sim.slopes()
    bx, by = _bits(sx, Lx).astype(np.int32), _bits(sy, Lx).astype(np.int32)
    assert np.all((2 * bx - 1).sum(axis=2) == 0)                    # every row closes periodically
    assert np.all((2 * by - 1).sum(axis=1) == 0)                    # every column too
    # curl-free on every plaquette: (x-1,y-1) -> (x,y) along x then y equals along y then x
    dx, dy = 2 * bx - 1, 2 * by - 1
    lhs = np.roll(dx, 1, axis=1) + np.roll(dy, 0, axis=1)           # dx[y-1][x] + dy[y][x]
    rhs = np.roll(dy, 1, axis=2) + dx                               # dy[y][x-1] + dx[y][x]
    assert np.array_equal(lhs, rhs)
    # heights: the oracle's row-0-then-columns path equals column-0-then-rows
    for s in range(S):
        h = sim.heights(s)
        alt = np.zeros_like(h)
        alt[0, 0] = dx[s, 0, 0]
        for y in range(1, Ly):
            alt[y, 0] = alt[y - 1, 0] + dy[s, y, 0]
        for x in range(1, Lx):
            alt[:, x] = alt[:, x - 1] + dx[s, :, x]
        assert np.array_equal(h, alt)
    assert np.all(sim.hops()[0] > 0)


def _histogram(sim, Lx, Ly):
    sx, sy = sim.slopes()
    bx, by = _bits(sx, Lx), _bits(sy, Lx)
    counts = {}
    for s in range(bx.shape[0]):
        key = (tuple(map(tuple, bx[s].tolist())), tuple(map(tuple, by[s].tolist())))
        counts[key] = counts.get(key, 0) + 1
    return counts


def _chi2(counts, dist, S):
    states = list(dist)
    exp = np.array([dist[k] * S for k in states])
    obs = np.array([counts.get(k, 0) for k in states], dtype=np.float64)
    stray = S - obs.sum()                                           # samples on states the distribution does not contain
    keep = exp >= 5
    c = ((obs[keep] - exp[keep]) ** 2 / exp[keep]).sum()
    if exp[~keep].sum() > 0:
        c += (obs[~keep].sum() - exp[~keep].sum()) ** 2 / exp[~keep].sum()
    return c + 1e6 * stray, int(keep.sum())


@pytest.mark.parametrize("p,q,mode", [(0.75, 0.25, "drawn"), (0.9, 0.3, "drawn"), (0.75, 0.25, "alternating")])
def test_finite_time_distribution_on_a_4x4_lattice_master_equation(p, q, mode):
    """Exact distribution after 2 MCS from the flat 4 x 4 surface (brute force, tests/master_equation.py) against the
    oracle's histogram over 30000 samples, plus the expected accepted moves.  Power: the same histogram rejects the
    other schedule, swapped p / q, and the reading "the x-pair alone decides"."""
    Lx = Ly = 4
    S, t = 30000, 2
    dist, fwd, bwd = ME.kpz2d_finite_time(Lx, Ly, p, q, t, mode)
    assert abs(sum(dist.values()) - 1.0) < 1e-12
    sim = R.Kpz2dRef(Lx, Ly, S, p, q, seed=77, offset_mode=1 if mode == "alternating" else 0)
    sim.run(t)
    counts = _histogram(sim, Lx, Ly)
    c, dof = _chi2(counts, dist, S)
    assert c < dof + 5 * np.sqrt(2 * dof), (c, dof)
    f, b = sim.hops()
    assert abs(f.mean() - fwd) < 5 * f.std(ddof=1) / np.sqrt(S)
    assert abs(b.mean() - bwd) < 5 * b.std(ddof=1) / np.sqrt(S) + 1e-12
    other = "alternating" if mode == "drawn" else "drawn"
    for alt in (ME.kpz2d_finite_time(Lx, Ly, p, q, t, other)[0], ME.kpz2d_finite_time(Lx, Ly, q, p, t, mode)[0]):
        assert _chi2(counts, alt, S)[0] > dof + 50 * np.sqrt(2 * dof)
    # "the x-pair alone decides" (no dimer constraint) after ONE MCS - its state space explodes at two
    one = R.Kpz2dRef(Lx, Ly, S, p, q, seed=78, offset_mode=1 if mode == "alternating" else 0)
    one.run(1)
    c1 = _histogram(one, Lx, Ly)
    good, dof1 = _chi2(c1, ME.kpz2d_finite_time(Lx, Ly, p, q, 1, mode)[0], S)
    assert good < dof1 + 5 * np.sqrt(2 * dof1), (good, dof1)
    assert _chi2(c1, ME.kpz2d_finite_time(Lx, Ly, p, q, 1, mode, need_both=False)[0], S)[0] > dof1 + 50 * np.sqrt(2 * dof1)


def test_particle_hole_symmetry_is_exact():
    """Inverting every slope maps forward-eligible sites onto backward-eligible ones; with p and q exchanged the same
    uniforms take the same decisions, so the two runs stay bitwise complements."""
    Lx, Ly, S = 12, 8, 4
    a = R.Kpz2dRef(Lx, Ly, S, 0.8, 0.3, seed=9)
    a.run(7)                                                        # some rough state
    sx, sy = a.slopes()
    mask = np.uint32((1 << Lx) - 1)
    b = R.Kpz2dRef(Lx, Ly, S, 0.3, 0.8, seed=9)
    b.set_slopes(~sx & mask, ~sy & mask)
    a2 = R.Kpz2dRef(Lx, Ly, S, 0.8, 0.3, seed=9)
    a2.set_slopes(sx, sy)
    a2.run(15)
    b.run(15)
    ax, ay = a2.slopes()
    bx, by = b.slopes()
    assert np.array_equal(bx, ~ax & mask) and np.array_equal(by, ~ay & mask)
    assert np.array_equal(a2.hops()[0], b.hops()[1])


def test_resume_and_first_sample_are_exact():
    Lx, Ly = 16, 8
    full = R.Kpz2dRef(Lx, Ly, 3, 0.75, 0.25, seed=3)
    full.set_record_times([4, 9])
    full.run(9)
    part = R.Kpz2dRef(Lx, Ly, 3, 0.75, 0.25, seed=3)
    part.set_record_times([4, 9])
    part.run(4)
    part.run(5)
    for x, y in zip(full.slopes(), part.slopes()):
        assert np.array_equal(x, y)
    assert np.array_equal(full.roughness()["sum_h2"], part.roughness()["sum_h2"])
    solo = R.Kpz2dRef(Lx, Ly, 1, 0.75, 0.25, seed=3, first_sample=2)
    solo.run(9)
    assert np.array_equal(solo.slopes()[0][0], full.slopes()[0][2])


def test_surface_roughens_slower_than_in_one_dimension():
    """2+1D KPZ: W^2 - 1/4 grows, with an effective exponent well below the 1+1D value 2 beta = 2/3 (the 2+1D KPZ value
    is 2 beta ~ 0.48; at these short times the crossover from the logarithmic Edwards-Wilkinson growth keeps it lower)."""
    L, S = 48, 6
    times = [4, 8, 16, 32, 64, 128]
    sim = R.Kpz2dRef(L, L, S, 0.75, 0.0, seed=21)
    sim.set_record_times(times)
    sim.run(times[-1])
    w2 = sim.roughness()["w2_mean"] - 0.25
    assert np.all(np.diff(w2) > 0)
    slope = np.polyfit(np.log(times[1:]), np.log(w2[1:]), 1)[0]
    assert 0.15 < slope < 0.55, slope
