"""GPU parity at the sizes the throughput claims are made on (VERDICT r1 "parity depth at full size").

The oracle needs minutes for these runs (it does ~2.6e7 site updates per second on one core), so its long jobs
start together in background threads when the first test of this module asks for one (the C library releases the GIL)
and every test waits for its own job only:

  job "config4"  L = 2^28, p = 0.9 / q = 0.1 (BASELINE.json configs[3]): 32 MCS from the flat start, lattice snapshots
                 at t = 1, 4, 32 and every record time up to 32 (a full 32-MCS chunk of the blocked path)     ~5 min
  job "config3"  sample S-1 of configs[2] alone, the full 10^5 MCS with all 50 records                          ~70 s
  job "config5"  sample S-1 of configs[4] alone, the full 10^5 MCS: state, currents, populations, profile       ~4 min
  job "2d-512"   sample S-1 of workload 2d-512 alone, the full 1000 MCS with all 20 records      ~2 min
  job "2d-1024"  sample S-1 of workload 2d-1024 alone, 100 MCS with the records up to there                      ~1 min

Run on the B200 box with:  python -m pytest tests -m gpu
"""
import concurrent.futures as cf

import numpy as np
import pytest

import workloads
from oracle import kpzref as R

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

C4_TIMES = [t for t in workloads.CONFIGS[4]["record_times"] if t < 32] + [32]
C4_SNAPSHOTS = (1, 4, 32)


@pytest.fixture(scope="module")
def K():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1012_0385_b200 as pkg
    pkg.load_library()
    return pkg


def _oracle_config4():
    c = workloads.CONFIGS[4]
    ref = R.KpzRef(c["L"], 1, c["p"], c["q"], seed=c["seed"])
    ref.set_record_times(C4_TIMES)
    out, t = {}, 0
    for stop in C4_SNAPSHOTS:
        ref.run(stop - t)
        t = stop
        out[stop] = ref.lattice().copy()
    out["rough"] = ref.roughness()
    ref.close()
    return out


def _oracle_config3():
    c = workloads.CONFIGS[3]
    ref = R.KpzRef(c["L"], 1, c["p"], c["q"], disorder=c["disorder"], seed=c["seed"], first_sample=c["S"] - 1)
    ref.set_record_times(c["record_times"])
    ref.run(c["n_mcs"])
    out = {"lattice": ref.lattice().copy(), "rough": ref.roughness(), "masks": ref.disorder_masks()}
    ref.close()
    return out


def _oracle_config5():
    c = workloads.CONFIGS[5]
    ref = R.LanesRef(c["L"], 1, c["p_a"], c["p_b"], c["rho0"], c["turn_prob"], c["turn_period"], c["omega"],
                     seed=c["seed"], first_sample=c["S"] - 1)
    ref.set_record_times(c["record_times"])
    ref.run(c["n_mcs"])
    out = {"state": [x.copy() for x in ref.state()], "cur": ref.currents(), "profile": ref.profile()}
    ref.close()
    return out


def _oracle_2d(key, n_mcs):
    c = workloads.CONFIGS[key]
    times = [t for t in c["record_times"] if t <= n_mcs]
    ref = R.Kpz2dRef(c["Lx"], c["Ly"], 1, c["p"], c["q"], seed=c["seed"], first_sample=c["S"] - 1)
    ref.set_record_times(times)
    ref.run(n_mcs)
    out = {"slopes": [x.copy() for x in ref.slopes()], "rough": ref.roughness(), "times": times}
    ref.close()
    return out


@pytest.fixture(scope="module")
def oracle_jobs():
    R.lib()                       # build / load once, before the threads start
    pool = cf.ThreadPoolExecutor(max_workers=5)
    jobs = {"config4": pool.submit(_oracle_config4), "config3": pool.submit(_oracle_config3),
            "config5": pool.submit(_oracle_config5), "2d-512": pool.submit(_oracle_2d, "2d-512", 1000),
            "2d-1024": pool.submit(_oracle_2d, "2d-1024", 100)}
    yield jobs
    pool.shutdown(wait=True)


# -----------------------------------------------------------------------------------------------------------------
# properties first: they need no oracle, the oracle jobs run meanwhile
# -----------------------------------------------------------------------------------------------------------------

def _torch_height_sums(words_i32, L):
    """Particle number, h_{L-1}, sum h and sum h^2 of one ring from its natural-layout words, by a plain torch prefix sum
    in pieces (independent of the library's reduction kernels)."""
    dev = words_i32.device
    shifts = torch.arange(32, device=dev, dtype=torch.int32)
    piece = 1 << 19                                      # words per piece = 2^24 sites
    carry = torch.zeros((), dtype=torch.int64, device=dev)
    n = torch.zeros((), dtype=torch.int64, device=dev)
    s1 = torch.zeros((), dtype=torch.int64, device=dev)
    s2 = torch.zeros((), dtype=torch.int64, device=dev)
    for w0 in range(0, L // 32, piece):
        w = words_i32[w0:w0 + piece]
        bits = ((w[:, None] >> shifts[None, :]) & 1).reshape(-1).to(torch.int64)
        n += bits.sum()
        h = torch.cumsum(2 * bits - 1, 0) + carry
        carry = h[-1].clone()
        s1 += h.sum()
        s2 += (h * h).sum()
    return int(n), int(carry), int(s1), int(s2)


def test_aux_ii_ring_of_2p32_sites_properties_and_k3_equals_k3t(K, oracle_jobs):
    """`4-aux-ii` (L = 2^32, the ring the HBM roofline is quoted on; "a single system by one card"): 8 MCS on
    the pass-by-pass kernel.  No oracle run is feasible (4 GiB of sites, ~3 min per MCS), so: particle number, h_{L-1} = 0,
    the library's exact sums against a plain torch prefix sum of the same lattice, and the blocked kernel (K3T), which
    shares no launch structure with it, reproducing the ring word for word."""
    c = workloads.CONFIGS["4-aux-ii"]
    L, n = c["L"], 8
    k3 = K.KpzSim(L, 1, c["p"], c["q"], seed=c["seed"], path=K.KPZ_PATH_STREAM, max_records=2)
    assert k3.path == K.KPZ_PATH_STREAM
    k3.set_record_times([3, n])
    k3.run(n)
    lat3 = k3.lattice()[0]
    npart, h_last, s1, s2 = _torch_height_sums(lat3, L)
    assert npart == L // 2 and h_last == 0
    r3 = k3.roughness()
    assert int(r3["sum_h"][1, 0]) == s1 and int(r3["sum_h2"][1, 0]) == s2
    assert 0.25 < r3["w2_mean"][1] < 10.0
    k3t = K.KpzSim(L, 1, c["p"], c["q"], seed=c["seed"], path=K.KPZ_PATH_BLOCKED, max_records=2)
    k3t.set_record_times([3, n])
    k3t.run(n)
    assert torch.equal(k3t.lattice()[0], lat3)
    rt = k3t.roughness()
    assert np.array_equal(rt["sum_h"], r3["sum_h"]) and np.array_equal(rt["sum_h2"], r3["sum_h2"])
    # the flat start is not a fixed point: the check above compares something that moved
    assert not torch.equal(lat3, torch.full_like(lat3, -0x55555556))


def test_config4_pass_by_pass_equals_blocked_for_40_mcs_at_full_size(K, oracle_jobs):
    c = workloads.CONFIGS[4]
    times = [t for t in c["record_times"] if t <= 40] + [40]
    sims = []
    for path in (K.KPZ_PATH_STREAM, K.KPZ_PATH_BLOCKED):
        g = K.KpzSim(c["L"], 1, c["p"], c["q"], seed=c["seed"], path=path, max_records=len(times))
        g.set_record_times(times)
        g.run(40)
        sims.append(g)
    assert torch.equal(sims[0].lattice(), sims[1].lattice())
    a, b = sims[0].roughness(), sims[1].roughness()
    assert np.array_equal(a["sum_h"], b["sum_h"]) and np.array_equal(a["sum_h2"], b["sum_h2"])


# -----------------------------------------------------------------------------------------------------------------
# against the oracle
# -----------------------------------------------------------------------------------------------------------------

def test_config3_last_sample_full_length(K, oracle_jobs):
    c = workloads.CONFIGS[3]
    gpu = K.KpzSim(c["L"], 1, c["p"], c["q"], disorder=c["disorder"], seed=c["seed"], first_sample=c["S"] - 1,
                   max_records=len(c["record_times"]))
    gpu.set_record_times(c["record_times"])
    gpu.run(c["n_mcs"])
    ref = oracle_jobs["config3"].result()
    gp, gq = gpu.disorder_masks()
    assert np.array_equal(K.words_to_numpy(gp), ref["masks"][0]) and np.array_equal(K.words_to_numpy(gq), ref["masks"][1])
    assert np.array_equal(K.words_to_numpy(gpu.lattice()), ref["lattice"])
    g, r = gpu.roughness(), ref["rough"]
    assert list(g["t"]) == list(r["t"]) == c["record_times"]
    assert np.array_equal(g["sum_h"], r["sum_h"]) and np.array_equal(g["sum_h2"], r["sum_h2"])


def test_config5_last_sample_full_length(K, oracle_jobs):
    c = workloads.CONFIGS[5]
    gpu = K.LanesSim(c["L"], 1, c["p_a"], c["p_b"], c["rho0"], c["turn_prob"], c["turn_period"], c["omega"],
                     seed=c["seed"], first_sample=c["S"] - 1, max_records=len(c["record_times"]))
    gpu.set_record_times(c["record_times"])
    gpu.run(c["n_mcs"])
    ref = oracle_jobs["config5"].result()
    for name, g, r in zip(("A", "B", "turn"), gpu.state(), ref["state"]):
        assert np.array_equal(K.words_to_numpy(g), r), name
    gc, rc = gpu.currents(), ref["cur"]
    assert list(gc["t"]) == list(rc["t"]) == c["record_times"]
    for key in ("j_a", "j_b", "n_a", "n_b"):
        assert np.array_equal(gc[key], rc[key]), key
    ga, gb, gn = gpu.profile()
    ra, rb, rn = ref["profile"]
    assert gn == rn == c["n_mcs"] // c["turn_period"]
    assert np.array_equal(K.words_to_numpy(ga), ra) and np.array_equal(K.words_to_numpy(gb), rb)


@pytest.mark.parametrize("path", ["blocked", "stream"])
def test_config4_full_size_against_oracle(K, oracle_jobs, path):
    """L = 2^28 against the oracle: the default blocked path for 32 MCS - one full chunk, records at every listed time
    up to 32 - and the pass-by-pass kernel for 4 MCS; lattice words at t = 1, 4 (and 32) and the exact sums."""
    c = workloads.CONFIGS[4]
    blocked = path == "blocked"
    stops = C4_SNAPSHOTS if blocked else C4_SNAPSHOTS[:2]
    times = [t for t in C4_TIMES if t <= stops[-1]]
    gpu = K.KpzSim(c["L"], 1, c["p"], c["q"], seed=c["seed"], max_records=len(times),
                   path=K.KPZ_PATH_BLOCKED if blocked else K.KPZ_PATH_STREAM)
    gpu.set_record_times(times)
    lats, t = {}, 0
    for stop in stops:
        gpu.run(stop - t)
        t = stop
        lats[stop] = gpu.lattice().clone()
    g = gpu.roughness()
    ref = oracle_jobs["config4"].result()
    for stop in stops:
        assert np.array_equal(K.words_to_numpy(lats[stop]), ref[stop]), f"lattice differs at t={stop}"
    r = ref["rough"]
    nt = len(times)
    assert list(g["t"]) == list(r["t"][:nt]) == times
    assert np.array_equal(g["sum_h"], r["sum_h"][:nt]) and np.array_equal(g["sum_h2"], r["sum_h2"][:nt])


@pytest.mark.parametrize("key,n_mcs", [("2d-512", 1000), ("2d-1024", 100)])
def test_2d_workloads_last_sample_in_the_full_launch(K, oracle_jobs, key, n_mcs):
    """The 2+1D bench workloads in their launch configuration (all samples: 256 CTAs of K5S / 64 clusters of 8 CTAs of
    K5C): the LAST sample against a solo oracle run - `2d-512` for its full 1000 MCS with all 20 records, `2d-1024` for
    100 MCS - slope words of both fields and the exact sums."""
    c = workloads.CONFIGS[key]
    times = [t for t in c["record_times"] if t <= n_mcs]
    gpu = K.Kpz2dSim(c["Lx"], c["Ly"], c["S"], c["p"], c["q"], seed=c["seed"], max_records=len(times))
    assert gpu.path == (K.KPZ_PATH_ONCHIP if key == "2d-512" else K.KPZ2D_PATH_CLUSTER)
    gpu.set_record_times(times)
    gpu.run(n_mcs)
    sx, sy = [K.words_to_numpy(t) for t in gpu.slopes()]
    g = gpu.roughness()
    ref = oracle_jobs[key].result()
    k = c["S"] - 1
    assert np.array_equal(sx[k], ref["slopes"][0][0]) and np.array_equal(sy[k], ref["slopes"][1][0])
    r = ref["rough"]
    assert list(g["t"]) == list(r["t"]) == times == ref["times"]
    assert np.array_equal(g["sum_h"][:, k], r["sum_h"][:, 0]) and np.array_equal(g["sum_h2"][:, k], r["sum_h2"][:, 0])
