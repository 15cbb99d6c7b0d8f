"""Brute-force master equation of the sub-lattice schedule on tiny rings (test helper, numpy only).

Independent of oracle/ and of the CUDA path: it enumerates states and builds the exact one-pass
transition matrices from the rule in PAPER.md:95 / DESIGN §R1-R3 (disjoint pairs (2j+o, 2j+o+1 mod L);
(1,0)->(0,1) w.p. p_a, (0,1)->(1,0) w.p. q_b), so a dropped term, a wrong rate site or a wrong pair set in
the oracle shows up as a disagreement with these numbers.
"""
from __future__ import annotations

import itertools

import numpy as np


def sector_states(L: int, N: int) -> list[int]:
    """All occupation bit patterns (bit i = n_i) with N particles on L sites."""
    return [sum(1 << i for i in c) for c in itertools.combinations(range(L), N)]


def pass_pairs(L: int, o: int) -> list[tuple[int, int]]:
    return [((2 * j + o) % L, (2 * j + o + 1) % L) for j in range(L // 2)]


def kpz_pass(L, states, o, p_site, q_site):
    """Exact transition matrix T[new, old] of one pass with offset o, and expected fwd/bwd hops per old state."""
    index = {s: k for k, s in enumerate(states)}
    n = len(states)
    T = np.zeros((n, n))
    fwd = np.zeros(n)
    bwd = np.zeros(n)
    for k, s in enumerate(states):
        outcomes = [(s, 1.0)]
        for a, b in pass_pairs(L, o):
            na, nb = (s >> a) & 1, (s >> b) & 1
            if na == 1 and nb == 0:
                r = p_site[a]
                fwd[k] += r
            elif na == 0 and nb == 1:
                r = q_site[b]
                bwd[k] += r
            else:
                continue
            flip = (1 << a) | (1 << b)
            nxt = []
            for st, pr in outcomes:
                if r > 0.0:
                    nxt.append((st ^ flip, pr * r))
                if r < 1.0:
                    nxt.append((st, pr * (1.0 - r)))
            outcomes = nxt
        for st, pr in outcomes:
            T[index[st], k] += pr
    return T, fwd, bwd


def stationary(K):
    """Stationary column vector of a column-stochastic matrix with a unique stationary state."""
    n = K.shape[0]
    A = K - np.eye(n)
    A[-1, :] = 1.0
    rhs = np.zeros(n)
    rhs[-1] = 1.0
    return np.linalg.solve(A, rhs)


def kpz_current_per_bond(L, N, p_site, q_site, mode):
    """Stationary net current per bond per MCS.  mode: 'drawn' (offset i.i.d. fair per pass) or 'alternating'."""
    states = sector_states(L, N)
    T0, f0, b0 = kpz_pass(L, states, 0, p_site, q_site)
    T1, f1, b1 = kpz_pass(L, states, 1, p_site, q_site)
    if mode == "drawn":
        K = 0.5 * (T0 + T1)
        pi = stationary(K)
        net = 0.5 * ((f0 - b0) + (f1 - b1))
        return 2.0 * float(pi @ net) / L
    if mode == "alternating":
        pi = stationary(T1 @ T0)
        return float(pi @ (f0 - b0) + (T0 @ pi) @ (f1 - b1)) / L
    raise ValueError(mode)


def kpz_finite_time(L, N, p_site, q_site, start_state, n_mcs, mode="drawn"):
    """Exact state distribution after n_mcs MCS from start_state, and expected accumulated fwd/bwd hops."""
    states = sector_states(L, N)
    T0, f0, b0 = kpz_pass(L, states, 0, p_site, q_site)
    T1, f1, b1 = kpz_pass(L, states, 1, p_site, q_site)
    v = np.zeros(len(states))
    v[states.index(start_state)] = 1.0
    fwd = bwd = 0.0
    for _ in range(n_mcs):
        for ps in (0, 1):
            if mode == "drawn":
                fwd += 0.5 * float(v @ (f0 + f1))
                bwd += 0.5 * float(v @ (b0 + b1))
                v = 0.5 * (T0 @ v + T1 @ v)
            else:
                T, f, b = (T0, f0, b0) if ps == 0 else (T1, f1, b1)
                fwd += float(v @ f)
                bwd += float(v @ b)
                v = T @ v
    return states, v, fwd, bwd


def width2(state: int, L: int) -> float:
    """W^2 of PAPER.md Eq. 3 for one configuration, heights = inclusive prefix of 2n-1 (plain floats)."""
    h = np.cumsum([2 * ((state >> i) & 1) - 1 for i in range(L)]).astype(float)
    return float(np.mean(h * h) - np.mean(h) ** 2)


# ---------------------------------------------------------------------------------------------------
# Two-lane model.  State = A bits | B bits << L.
# ---------------------------------------------------------------------------------------------------

def lanes_states(L, NT):
    """All (A,B) patterns with N_A + N_B = NT."""
    out = []
    for s in range(1 << (2 * L)):
        if bin(s).count("1") == NT:
            out.append(s)
    return out


def lanes_pass(L, states, o, p_a, p_b):
    """In-lane pass of both lanes with the same offset: A hops right (a->b), B hops left (b->a)."""
    index = {s: k for k, s in enumerate(states)}
    n = len(states)
    T = np.zeros((n, n))
    ja = np.zeros(n)
    jb = np.zeros(n)
    for k, s in enumerate(states):
        A, B = s & ((1 << L) - 1), s >> L
        outcomes = [(s, 1.0)]
        for a, b in pass_pairs(L, o):
            moves = []
            if (A >> a) & 1 == 1 and (A >> b) & 1 == 0:
                ja[k] += p_a
                moves.append(((1 << a) | (1 << b), p_a))
            if (B >> a) & 1 == 0 and (B >> b) & 1 == 1:
                jb[k] += p_b
                moves.append((((1 << a) | (1 << b)) << L, p_b))
            for flip, r in moves:
                nxt = []
                for st, pr in outcomes:
                    if r > 0.0:
                        nxt.append((st ^ flip, pr * r))
                    if r < 1.0:
                        nxt.append((st, pr * (1.0 - r)))
                outcomes = nxt
        for st, pr in outcomes:
            T[index[st], k] += pr
    return T, ja, jb


def lanes_switch(L, states, turn_mask, omega, a_to_b, w_unflagged=0.0):
    """Crossing probability omega at the sites of turn_mask, w_unflagged elsewhere (0: turning-point model)."""
    index = {s: k for k, s in enumerate(states)}
    n = len(states)
    T = np.zeros((n, n))
    for k, s in enumerate(states):
        A, B = s & ((1 << L) - 1), s >> L
        outcomes = [(s, 1.0)]
        for i in range(L):
            w = omega if (turn_mask >> i) & 1 else w_unflagged
            src, dst = (A, B) if a_to_b else (B, A)
            if (src >> i) & 1 == 1 and (dst >> i) & 1 == 0:
                flip = (1 << i) | (1 << (i + L))
                nxt = []
                for st, pr in outcomes:
                    if w > 0.0:
                        nxt.append((st ^ flip, pr * w))
                    if w < 1.0:
                        nxt.append((st, pr * (1.0 - w)))
                outcomes = nxt
        for st, pr in outcomes:
            T[index[st], k] += pr
    return T


def lanes_finite_time(L, start_state, turn_mask, p_a, p_b, omega, n_mcs, ab_first=True, w_unflagged=0.0,
                      mask_v=None):
    """Exact distribution and expected J_A, J_B after n_mcs MCS (drawn offsets, fixed turn mask).
    ab_first=False swaps the two lane-change steps (an alternative reading used to show test power)."""
    NT = bin(start_state).count("1")
    states = lanes_states(L, NT)
    T0, ja0, jb0 = lanes_pass(L, states, 0, p_a, p_b)
    T1, ja1, jb1 = lanes_pass(L, states, 1, p_a, p_b)
    SAB = lanes_switch(L, states, turn_mask, omega, True, w_unflagged)
    SBA = lanes_switch(L, states, turn_mask if mask_v is None else mask_v, omega, False, w_unflagged)
    v = np.zeros(len(states))
    v[states.index(start_state)] = 1.0
    JA = JB = 0.0
    for _ in range(n_mcs):
        for S in ((SAB, SBA) if ab_first else (SBA, SAB)):
            JA += 0.5 * float(v @ (ja0 + ja1))
            JB += 0.5 * float(v @ (jb0 + jb1))
            v = 0.5 * (T0 @ v + T1 @ v)
            v = S @ v
    return states, v, JA, JB


# ------------------------------------------------------------------------------------------------
# 2+1D generalisation: checkerboard passes of the dimer / octahedron move on a tiny
# periodic Lx x Ly lattice.  A state is (sx, sy), two tuples of Ly rows of Lx bits; written without reference to the
# oracle: site (x, y), colour (x + y) & 1; forward move iff x-pair and y-pair are both (1,0), backward iff both (0,1).
# ------------------------------------------------------------------------------------------------
def flat2d(Lx, Ly):
    rows = tuple(tuple((x + y) & 1 for x in range(Lx)) for y in range(Ly))
    return rows, rows


def _moves2d(state, Lx, Ly, colour, need_both=True):
    """Eligible moves of one colour pass: list of (x, y, kind) with kind +1 forward, -1 backward."""
    sx, sy = state
    out = []
    for y in range(Ly):
        for x in range(Lx):
            if (x + y) & 1 != colour:
                continue
            xp = (sx[y][x], sx[y][(x + 1) % Lx])
            yp = (sy[y][x], sy[(y + 1) % Ly][x])
            if need_both:
                if xp == (1, 0) and yp == (1, 0):
                    out.append((x, y, +1))
                elif xp == (0, 1) and yp == (0, 1):
                    out.append((x, y, -1))
            else:                       # a WRONG reading kept for the power check: the x-pair alone decides
                if xp == (1, 0):
                    out.append((x, y, +1))
                elif xp == (0, 1):
                    out.append((x, y, -1))
    return out


def _apply2d(state, Lx, Ly, chosen):
    sx = [list(r) for r in state[0]]
    sy = [list(r) for r in state[1]]
    for x, y, kind in chosen:
        a, b = (0, 1) if kind > 0 else (1, 0)
        sx[y][x], sx[y][(x + 1) % Lx] = a, b
        sy[y][x], sy[(y + 1) % Ly][x] = a, b
    return tuple(tuple(r) for r in sx), tuple(tuple(r) for r in sy)


def kpz2d_finite_time(Lx, Ly, p, q, n_mcs, mode="drawn", need_both=True):
    """Exact distribution {state: probability} after n_mcs MCS from the flat state, and the expected numbers of accepted
    forward / backward moves.  mode "drawn": every pass has colour 0 or 1 with probability 1/2; "alternating": 0 then 1."""
    import itertools
    dist = {flat2d(Lx, Ly): 1.0}
    fwd = bwd = 0.0
    for _ in range(n_mcs):
        for ps in range(2):
            new = {}
            colours = [(0, 0.5), (1, 0.5)] if mode == "drawn" else [(ps, 1.0)]
            for state, pr in dist.items():
                for colour, pc in colours:
                    mv = _moves2d(state, Lx, Ly, colour, need_both)
                    for pick in itertools.product((0, 1), repeat=len(mv)):
                        w = pr * pc
                        chosen = []
                        for take, (x, y, kind) in zip(pick, mv):
                            rate = p if kind > 0 else q
                            w *= rate if take else 1.0 - rate
                            if take:
                                chosen.append((x, y, kind))
                        if w == 0.0:
                            continue
                        fwd += w * sum(1 for c in chosen if c[2] > 0)
                        bwd += w * sum(1 for c in chosen if c[2] < 0)
                        ns = _apply2d(state, Lx, Ly, chosen)
                        new[ns] = new.get(ns, 0.0) + w
            dist = new
    return dist, fwd, bwd
