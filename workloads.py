"""Seeded synthetic workloads — the five BASELINE.json configs as plain parameter sets.

This module is the ONLY thing the CUDA path's callers and the oracle's callers share.  It holds no
arithmetic of the method (no Philox, no update rule, no heights): just sizes, probabilities, seeds and the
integer record-time lists.  Everything else (initial lattices, disorder masks, turning points) is derived
from the seed independently by each implementation.

Record times: t_0 = 1, t_k = max(t_{k-1}+1, floor(T^(k/(K-1)) + 0.5)), last forced to T.
The lists below are frozen literals; tests/test_workloads.py checks the rule reproduces them.
"""
from __future__ import annotations

import math


def log_spaced_times(T: int, K: int) -> list[int]:
    ts = [1]
    for k in range(1, K):
        v = int(math.floor(T ** (k / (K - 1)) + 0.5))
        ts.append(max(ts[-1] + 1, v))
    ts[-1] = T
    return ts


_T40_1E4 = [1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 13, 17, 22, 27, 35, 44, 55, 70, 89, 113, 143, 180, 229, 289, 367,
            464, 588, 744, 943, 1194, 1512, 1914, 2424, 3070, 3888, 4924, 6236, 7897, 10000]
_T50_1E5 = [1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 13, 17, 21, 27, 34, 43, 54, 69, 87, 110, 139, 176, 222, 281, 356,
            450, 569, 720, 910, 1151, 1456, 1842, 2330, 2947, 3728, 4715, 5964, 7543, 9541, 12068, 15264, 19307,
            24421, 30888, 39069, 49417, 62506, 79060, 100000]
_T20_1E3 = [1, 2, 3, 4, 5, 6, 9, 13, 18, 26, 38, 55, 78, 113, 162, 234, 336, 483, 695, 1000]

def eq7_times(T: int, t0: int = 30, factor: float = 1.05) -> list[int]:
    """The paper's sampling times, Eq. 7: t_0 = 30, t_{i+1} = 1.05 t_i, made integer and strictly
    increasing: t_{i+1} = max(t_i + 1, floor(1.05 t_i)); times beyond T are dropped."""
    ts, t = [], t0
    while t <= T:
        ts.append(t)
        t = max(t + 1, int(math.floor(t * factor)))
    return ts


# BASELINE.json `configs`[0..4]  (numbered 1..5 as in SURVEY.md §8(d)).
CONFIGS = {
    1: dict(name="config1_kpz_L64_S16_p1", kind="kpz", L=64, S=16, p=1.0, q=0.0, disorder=None, n_mcs=1000,
            record_times=[1, 2, 4, 8, 16, 32, 64, 128, 256, 512, 1000], seed=1),
    2: dict(name="config2_kpz_L8192_S1024_p075_q025", kind="kpz", L=8192, S=1024, p=0.75, q=0.25, disorder=None,
            n_mcs=10_000, record_times=_T40_1E4, seed=2),
    # disorder = (prob_slow_p, p_slow, prob_slow_q, q_slow)
    3: dict(name="config3_disorder_L16384_S512", kind="kpz", L=16384, S=512, p=1.0, q=0.0,
            disorder=(0.1, 0.5, 0.0, 0.0), n_mcs=100_000, record_times=_T50_1E5, seed=3),
    4: dict(name="config4_stream_L2p28_S1_p09_q01", kind="kpz", L=1 << 28, S=1, p=0.9, q=0.1, disorder=None,
            n_mcs=1000, record_times=_T20_1E3, seed=4),
    5: dict(name="config5_lanes_L16384_S256", kind="lanes", L=16384, S=256, p_a=1.0, p_b=1.0, rho0=0.3,
            turn_prob=0.05, turn_period=100, omega=0.1, n_mcs=100_000, record_times=_T50_1E5, seed=5),
    # Configs 2 and 3 with sample counts that fill a B200's warp slots evenly (592 SMSPs x 2 resp. 4 warps): the
    # BASELINE.json counts (1024 one-warp rings, 512 two-warp rings) leave 13.5 % of the second slots empty.
    "2-fill": dict(name="config2_shape_S1184", kind="kpz", L=8192, S=1184, p=0.75, q=0.25, disorder=None,
                   n_mcs=10_000, record_times=_T40_1E4, seed=2),
    "3-fill": dict(name="config3_shape_S1184", kind="kpz", L=16384, S=1184, p=1.0, q=0.0,
                   disorder=(0.1, 0.5, 0.0, 0.0), n_mcs=20_000, record_times=[t for t in _T50_1E5 if t <= 20_000] + [20_000],
                   seed=3),
    # Auxiliary streamed runs: dyadic rates, the pass-by-pass streamed kernel (path 2) forced, so
    # that the sweep is bandwidth-bound: (i) ring in L2, (ii) ring beyond L2 (the HBM roofline case).
    "4-aux-i": dict(name="config4aux1_stream_L2p28_p075_q025", kind="kpz", L=1 << 28, S=1, p=0.75, q=0.25,
                    disorder=None, n_mcs=1000, record_times=_T20_1E3, seed=4, path=2),
    "4-aux-ii": dict(name="config4aux2_stream_L2p32_p075_q025", kind="kpz", L=1 << 32, S=1, p=0.75, q=0.25,
                     disorder=None, n_mcs=200, record_times=[1, 2, 4, 8, 16, 32, 64, 128, 200], seed=4, path=2),
    # the paper's own parameter sets on the same kernels: TASEP p=0.8, q=0, strict
    # even/odd alternation (offset_mode 1), Eq. 7 sampling.  "paper-1024x30" is the launch the paper times (30
    # realisations of L=1024 to 10^6 MCS in 4.2 s on a Quadro FX 5800 = 7.3 GSU/s); "paper-1024-fill" is the same ring
    # with enough realisations to fill a B200 (2 warps per SMSP, 8 rings per warp).
    "paper-1024x30": dict(name="paper_tasep_L1024_S30_p08", kind="kpz", L=1024, S=30, p=0.8, q=0.0, disorder=None,
                          n_mcs=1_000_000, record_times=eq7_times(1_000_000), seed=6, offset_mode=1,
                          paper_gsu=30 * 1024 * 1e6 / 4.2 / 1e9),
    "paper-1024-fill": dict(name="paper_tasep_L1024_S9472_p08", kind="kpz", L=1024, S=9472, p=0.8, q=0.0,
                            disorder=None, n_mcs=10_000, record_times=eq7_times(10_000), seed=6, offset_mode=1),
    # Q-TASEP (Eq. 8): Q = 0.5, slow sites hop with r p, r = 0.5 (the paper does not state r here)
    "paper-qtasep-16384": dict(name="paper_qtasep_L16384_S512", kind="kpz", L=16384, S=512, p=0.8, q=0.0,
                               disorder=(0.5, 0.4, 0.0, 0.0), n_mcs=10_000, record_times=eq7_times(10_000), seed=7,
                               offset_mode=1),
    # Q-SSEP: p = q with disorder r = 0.2 on both rates, L = 4096
    "paper-qssep-4096": dict(name="paper_qssep_L4096_S2048", kind="kpz", L=4096, S=2048, p=0.5, q=0.5,
                             disorder=(0.5, 0.1, 0.5, 0.1), n_mcs=10_000, record_times=eq7_times(10_000), seed=8,
                             offset_mode=1),
    # the paper's own two-lane model: in-lane p = 0.5, half filling, every site crossed
    # with 0.8 (0.2 at sites flagged with probability 1/2), separate quenched flags u_i, v_i, L = 4096, Eq. 7 sampling
    "paper-lanes-4096": dict(name="paper_two_lane_L4096_S1024", kind="lanes", L=4096, S=1024, p_a=0.5, p_b=0.5, rho0=0.5,
                             turn_prob=0.5, turn_period=0, omega=0.2, w_unflagged=0.8, independent=1, n_mcs=10_000,
                             record_times=eq7_times(10_000), seed=9, offset_mode=1),
    # PAPER.md:235-239 (Sect. 2.4, Fig. 8a): "running the simulations up to t_max = 10^5 MCs for 560 realizations" of
    # the TASEP for 512 <= L <= 32K; the paper reports T ~ L^0.9 on a Tesla C2070.  Keys "paper-scan-512" ... "-32768"
    # are added below (`_add_scan`).
    # the same two rings on the default (temporally blocked) path
    "4-aux-i-blocked": dict(name="config4aux1_blocked_L2p28_p075_q025", kind="kpz", L=1 << 28, S=1, p=0.75, q=0.25,
                            disorder=None, n_mcs=1000, record_times=_T20_1E3, seed=4),
}


# the 2+1D generalisation: 64 independent 1024 x 1024 surfaces of the dimer
# / octahedron model, p = 0.75, q = 0, 1000 MCS, 20 log-spaced record times.  "site updates" = Lx * Ly per MCS and sample.
CONFIGS["2d-512"] = dict(name="kpz2d_L512x512_S256_p075", kind="kpz2d", Lx=512, Ly=512, L=512 * 512, S=256, p=0.75, q=0.0,
                         n_mcs=1000, record_times=_T20_1E3, seed=12)   # a sample (64 KiB of slopes) stays in shared memory
CONFIGS["2d-1024"] = dict(name="kpz2d_L1024x1024_S64_p075", kind="kpz2d", Lx=1024, Ly=1024, L=1024 * 1024, S=64, p=0.75,
                          q=0.0, n_mcs=1000, record_times=_T20_1E3, seed=12)
# 16 surfaces of 2048 x 2048 (1 MiB of slopes each): a sample over a cluster of 16 CTAs (the non-portable cluster size)
CONFIGS["2d-2048"] = dict(name="kpz2d_L2048x2048_S16_p075", kind="kpz2d", Lx=2048, Ly=2048, L=2048 * 2048, S=16, p=0.75,
                          q=0.0, n_mcs=1000, record_times=_T20_1E3, seed=12)
# one surface of 32768 x 32768 (2^30 sites, 512 MiB of slope planes): beyond the L2 and every on-chip variant - the streamed
# kernel K5, one launch per colour pass, against the HBM roofline (1 byte per site update: every plane word is read once
# and written once per pass)
CONFIGS["2d-32768"] = dict(name="kpz2d_L32768x32768_S1_p075", kind="kpz2d", Lx=32768, Ly=32768, L=32768 * 32768, S=1, p=0.75,
                           q=0.0, n_mcs=20, record_times=[4, 20], seed=12, no_cpu_baseline="one MCS of this lattice takes the "
                           "oracle about 8 minutes")
# the same 512 x 512 ensemble with every sample spread over a thread-block cluster (K5C; options.path = 3): smaller CTAs,
# which balance better over 148 SMs
CONFIGS["2d-512-cluster"] = dict(CONFIGS["2d-512"], name="kpz2d_L512x512_S256_p075_cluster", path=3)


def _add_scan() -> None:
    for k in range(9, 16):
        L = 1 << k
        CONFIGS[f"paper-scan-{L}"] = dict(name=f"paper_scan_tasep_L{L}_S560_p08", kind="kpz", L=L, S=560, p=0.8, q=0.0,
                                          disorder=None, n_mcs=100_000, record_times=eq7_times(100_000), seed=10,
                                          offset_mode=1)


_add_scan()


def site_updates(cfg: dict, n_mcs: int | None = None, nsamples: int | None = None) -> int:
    """Site updates of a run: L per MCS per sample; the two-lane model counts both lanes."""
    n = cfg["n_mcs"] if n_mcs is None else n_mcs
    s = cfg["S"] if nsamples is None else nsamples
    lanes = 2 if cfg["kind"] == "lanes" else 1
    return lanes * cfg["L"] * s * n


def truncated(cfg: dict, n_mcs: int, nsamples: int | None = None, first_sample: int = 0) -> dict:
    """The same workload cut to n_mcs steps / nsamples samples starting at global sample `first_sample`."""
    c = dict(cfg)
    c["n_mcs"] = n_mcs
    c["record_times"] = [t for t in cfg["record_times"] if t <= n_mcs]
    if nsamples is not None:
        c["S"] = nsamples
    c["first_sample"] = first_sample
    return c
