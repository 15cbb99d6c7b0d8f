"""GPU parity of the 2+1D generalisation: kernel K5 through the C ABI
against the CPU oracle, bit for bit - slope words of both fields, int32 heights, exact sums - plus properties at a size
the oracle cannot reach.

Run on the B200 box with:  python -m pytest tests -m gpu
"""
import numpy as np
import pytest

import workloads
from oracle import kpzref as R

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def K():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1012_0385_b200 as pkg
    pkg.load_library()
    return pkg


def run_both_2d(K, Lx, Ly, S, p, q, seed, times, chunks, first_sample=0, offset_mode=0, start=None, path=0):
    if isinstance(path, tuple):          # (path, kpz_debug_config spec): see PATHS
        with K.debug_config(path[1]):
            return run_both_2d(K, Lx, Ly, S, p, q, seed, times, chunks, first_sample, offset_mode, start, path[0])
    total = sum(chunks)
    times = [t for t in times if t <= total]
    try:
        gpu = K.Kpz2dSim(Lx, Ly, S, p, q, seed=seed, first_sample=first_sample, offset_mode=offset_mode,
                         max_records=max(len(times), 1), path=path)
    except K.KpzError as e:
        if path == K.KPZ2D_PATH_CLUSTER and e.code == -2:
            pytest.skip("no cluster shape for this lattice")      # Lx % 256, Ly % (2 CS): refused, not mis-run
        raise
    ref = R.Kpz2dRef(Lx, Ly, S, p, q, seed=seed, first_sample=first_sample, offset_mode=offset_mode)
    if path:
        assert gpu.path == path
    if start is not None:
        ref.set_slopes(*start)
        gpu.set_slopes(K.words_from_numpy(start[0], gpu.device), K.words_from_numpy(start[1], gpu.device))
    ref.set_record_times(times)
    gpu.set_record_times(times)

    def same(tag):
        for name, g, r in zip(("sx", "sy"), gpu.slopes(), ref.slopes()):
            assert np.array_equal(K.words_to_numpy(g), r), f"{name} differs {tag}"
    same("initially")
    done = 0
    for n in chunks:
        ref.run(n)
        gpu.run(n)
        done += n
        assert gpu.time == ref.time == done
        same(f"at t={done}")
    g, r = gpu.roughness(), ref.roughness()
    assert list(g["t"]) == list(r["t"]) == times
    assert np.array_equal(g["sum_h"], r["sum_h"]) and np.array_equal(g["sum_h2"], r["sum_h2"])
    assert np.array_equal(g["w2_mean"], r["w2_mean"]) or np.allclose(g["w2_mean"], r["w2_mean"], rtol=1e-15, atol=0)
    for s in (0, S - 1):
        assert np.array_equal(gpu.heights(s).cpu().numpy(), ref.heights(s)), f"heights of sample {s} differ"
    return gpu, g


# 1 = a sample in shared memory (K5S), 2 = one launch per colour pass (K5); each as the run-time specialised kernel
# (NVRTC: shape and thresholds are constants) and as the generic kernel of the library build ("jit=0"); K5J_RIW=0 takes
# the shuffles out of the specialised on-chip kernel (neighbour word loaded, carries by atomics), K5J_PIPE=0 its
# software pipeline (planes drawn one sweep ahead around a split barrier)
# K5J_PDL=0: consecutive passes of the streamed kernel launched without programmatic dependent launch
# 3 = a sample spread over a thread-block cluster (K5C; 2 CTAs unless K5J_CS forces 4, 8 or 16), rows of the neighbour CTA
# through distributed shared memory, one barrier.cluster per pass (K5J_NBR=1: the CTAs synchronise with their two neighbours
# only, through mbarriers); shapes without a cluster decomposition are refused (and skipped here)
PATHS = [(1, ""), (2, ""), (2, "K5J_PDL=0"), (1, "jit=0"), (2, "jit=0"), (1, "K5J_RIW=0"), (1, "K5J_PIPE=0"), (3, ""), (3, "K5J_CS=4"),
         (3, "K5J_CS=8"), (3, "K5J_CS=16"), (3, "K5J_RIW=0"), (3, "K5J_NBR=1"), (3, "K5J_DUAL=1"), (3, "K5J_DUAL=1;K5J_CS=4")]


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("Lx,Ly", [(64, 2), (64, 6), (128, 64), (192, 10), (256, 256), (320, 30), (1024, 4), (256, 2), (512, 64),
                                   (768, 6), (2048, 8), (8192, 2), (16384, 2), (512, 130), (768, 48), (256, 16), (1024, 32), (16384, 8), (2048, 64)])
def test_sizes_ragged_supergroups_and_tiny_lattices(K, Lx, Ly, path):
    """A row of 64 sites is a quarter of a Philox supergroup, 192 / 320 sites leave ragged ones; Ly = 2 couples every row
    to itself through the periodic y-pair; 256 x 256 gives the 512 threads of the on-chip kernel one supergroup each.
    Fast path (Lx a multiple of 256, threads taken by row parity): 512 x 64, 2048 x 8 and 8192 x 2 keep a row inside a
    warp (2, 8, 32 lanes: shuffles), 768 x 6 has three supergroups per row and warps of mixed colour on the streamed
    path, 16384 x 2 rows longer than a warp, 512 x 130 a last warp that is partly idle."""
    run_both_2d(K, Lx, Ly, 3, 0.75, 0.25, seed=Lx + Ly, times=[1, 3, 12], chunks=[5, 7], path=path)


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("p,q", [(1.0, 0.0), (0.0, 1.0), (0.5, 0.5), (0.9, 0.1), (0.3, 0.6), (1.0, 1.0), (0.0, 0.0), (0.8, 0.0)])
def test_rate_classes(K, p, q, path):
    run_both_2d(K, 128, 32, 2, p, q, seed=7, times=[2, 9], chunks=[9], path=path)


@pytest.mark.parametrize("path", PATHS)
def test_alternating_colours_resume_first_sample_and_rough_start(K, path):
    run_both_2d(K, 128, 16, 2, 0.75, 0.25, seed=9, times=[4, 11], chunks=[3, 1, 7], offset_mode=1, path=path)
    run_both_2d(K, 128, 16, 1, 0.75, 0.25, seed=9, times=[11], chunks=[11], first_sample=5, path=path)
    rough = R.Kpz2dRef(64, 8, 2, 0.6, 0.4, seed=1)
    rough.run(25)
    run_both_2d(K, 64, 8, 2, 0.2, 0.9, seed=3, times=[6], chunks=[6], start=rough.slopes(), path=path)


@pytest.mark.parametrize("path", PATHS)
def test_fast_path_alternating_colours_first_sample_and_rough_start(K, path):
    """The same on a lattice every kernel takes on its fast path (Lx = 512: K5S pipeline, K5C clusters): alternating
    colours, a resumed run, a handle that starts at global sample 5, a rough start handed in through kpz2d_set_slopes."""
    run_both_2d(K, 512, 32, 2, 0.75, 0.25, seed=9, times=[4, 11], chunks=[3, 1, 7], offset_mode=1, path=path)
    run_both_2d(K, 512, 32, 1, 0.75, 0.0, seed=9, times=[11], chunks=[11], first_sample=5, path=path)
    rough = R.Kpz2dRef(512, 32, 3, 0.6, 0.4, seed=1)
    rough.run(25)
    run_both_2d(K, 512, 32, 3, 0.2, 0.9, seed=3, times=[6, 18], chunks=[6, 12], start=rough.slopes(), path=path)


@pytest.mark.parametrize("path", PATHS)
def test_offset_batches_and_chunks_are_crossed(K, path):
    """kpz2d_run draws the colour offsets for 1024 passes (512 MCS) at a time on the streamed path, for 16 MCS at a time in
    the on-chip kernel: one run across those boundaries, records on and around them."""
    run_both_2d(K, 64, 4, 2, 0.75, 0.25, seed=13, times=[15, 16, 17, 511, 512, 513, 1100], chunks=[1100], path=path)


def test_path_selection_and_both_paths_agree_at_512(K):
    a = K.Kpz2dSim(512, 512, 2, 0.75, 0.0, seed=5, max_records=1)
    assert a.path == K.KPZ_PATH_ONCHIP                             # 64 KiB of slopes per sample
    b = K.Kpz2dSim(512, 512, 2, 0.75, 0.0, seed=5, max_records=1, path=K.KPZ_PATH_STREAM)
    assert K.Kpz2dSim(1024, 1024, 1, 0.75, 0.0, seed=5, max_records=1).path == K.KPZ2D_PATH_CLUSTER   # 256 KiB: 4 CTAs
    with K.debug_config("jit=0"):
        assert K.Kpz2dSim(1024, 1024, 1, 0.75, 0.0, seed=5, max_records=1).path == K.KPZ_PATH_STREAM
    assert K.Kpz2dSim(2048, 2048, 1, 0.75, 0.0, seed=5, max_records=1).path == K.KPZ2D_PATH_CLUSTER       # 1 MiB: 16 CTAs
    assert K.Kpz2dSim(4096, 4096, 1, 0.75, 0.0, seed=5, max_records=1).path == K.KPZ_PATH_STREAM           # 4 MiB
    assert K.Kpz2dSim(1024, 1022, 1, 0.75, 0.0, seed=5, max_records=1).path == K.KPZ_PATH_STREAM           # rows do not divide
    with pytest.raises(K.KpzError):
        K.Kpz2dSim(2048, 2048, 1, 0.75, 0.0, seed=5, max_records=1, path=K.KPZ_PATH_ONCHIP)
    c = K.Kpz2dSim(512, 512, 2, 0.75, 0.0, seed=5, max_records=1, path=K.KPZ2D_PATH_CLUSTER)
    for g in (a, b, c):
        g.set_record_times([40])
        g.run(40)
    for other in (b, c):
        for x, y in zip(a.slopes(), other.slopes()):
            assert torch.equal(x, y)
        ra, rb = a.roughness(), other.roughness()
        assert np.array_equal(ra["sum_h"], rb["sum_h"]) and np.array_equal(ra["sum_h2"], rb["sum_h2"])


@pytest.mark.parametrize("spec", ["", "jit=0", "K5J_CS=8"])
@pytest.mark.parametrize("key", ["2d-512", "2d-1024"])
def test_workload_shape_sampled_against_solo_oracle_runs(K, key, spec):
    """The bench workloads `2d-512` (on chip) and `2d-1024` (over a cluster; streamed with jit=0) in their launch configuration (all samples),
    shortened: first and last sample against solo oracle runs, every sample single-valued."""
    c = workloads.CONFIGS[key]
    n, times = 6, [1, 2, 3, 4, 5, 6]
    with K.debug_config(spec):
        gpu = K.Kpz2dSim(c["Lx"], c["Ly"], c["S"], c["p"], c["q"], seed=c["seed"], max_records=len(times))
        gpu.set_record_times(times)
        gpu.run(n)
    sx, sy = [K.words_to_numpy(t) for t in gpu.slopes()]
    r = gpu.roughness()
    for k in (0, c["S"] - 1):
        ref = R.Kpz2dRef(c["Lx"], c["Ly"], 1, c["p"], c["q"], seed=c["seed"], first_sample=k)
        ref.set_record_times(times)
        ref.run(n)
        rx, ry = ref.slopes()
        assert np.array_equal(sx[k], rx[0]) and np.array_equal(sy[k], ry[0])
        rr = ref.roughness()
        assert np.array_equal(r["sum_h"][:, k], rr["sum_h"][:, 0]) and np.array_equal(r["sum_h2"][:, k], rr["sum_h2"][:, 0])
    bits = np.unpackbits(sx.view(np.uint8), bitorder="little").reshape(c["S"], c["Ly"], c["Lx"])
    assert np.all(bits.sum(axis=2) == c["Lx"] // 2)                 # every row closes periodically
    bits = np.unpackbits(sy.view(np.uint8), bitorder="little").reshape(c["S"], c["Ly"], c["Lx"])
    assert np.all(bits.sum(axis=1) == c["Ly"] // 2)                 # every column too


def test_growth_at_a_size_the_oracle_cannot_reach(K):
    """2+1D KPZ (refs. [7, 28] of the paper): W^2 - 1/4 grows with an effective exponent 2 beta well below the 1+1D 2/3;
    the exact sums of kpz2d_roughness equal a torch reduction of kpz2d_heights."""
    L, S = 1024, 4
    times = [2 ** k for k in range(2, 11)]
    gpu = K.Kpz2dSim(L, L, S, 0.75, 0.0, seed=31, max_records=len(times))
    gpu.set_record_times(times)
    gpu.run(times[-1])
    r = gpu.roughness()
    h = gpu.heights(S - 1).to(torch.int64)
    assert int(h.sum()) == r["sum_h"][-1, S - 1] and int((h * h).sum()) == r["sum_h2"][-1, S - 1]
    w2 = r["w2_mean"] - 0.25
    assert np.all(np.diff(w2) > 0)
    local = np.diff(np.log(w2)) / np.diff(np.log(np.array(times, dtype=np.float64)))
    assert np.all((local[3:] > 0.2) & (local[3:] < 0.6)), local


def test_growth_exponents_kpz_and_edwards_wilkinson_classes(K):
    """Physics of the reading R19 at a size and statistics the kernels make cheap (256 surfaces of 512 x 512, 4096 MCS in
    half a second): with a bias (p = 0.75, q = 0) the octahedron model is in the 2+1D KPZ class - refs. [7, 28] of the
    paper report beta ~ 0.24, W^2 - 1/4 ~ t^0.48 - while the unbiased model (p = q) is in the
    Edwards-Wilkinson class, whose width grows only logarithmically in two dimensions: the local exponent decays."""
    from paper_1012_0385_b200 import analysis
    times = [2 ** k for k in range(2, 13)]
    out = {}
    for name, p, q, seed in (("kpz", 0.75, 0.0, 12), ("ew", 0.5, 0.5, 3)):
        g = K.Kpz2dSim(512, 512, 256, p, q, seed=seed, max_records=len(times))
        g.set_record_times(times)
        g.run(times[-1])
        r = g.roughness()
        out[name] = analysis.local_exponents(r["t"], r["w2_mean"] - 0.25), r["w2_mean"]
    t = np.array(times, dtype=np.float64)
    sel = (t >= 128) & (t <= 2048)                     # past the early transient, before L = 512 is felt
    two_beta = np.polyfit(np.log(t[sel]), np.log(out["kpz"][1][sel] - 0.25), 1)[0]
    assert 0.43 < two_beta < 0.51, two_beta            # measured 0.46 ... 0.47 (effective; asymptotically 0.48)
    ew = out["ew"][0]
    assert np.all(np.diff(ew[2:]) < 0.0) and ew[-1] < 0.15, ew      # measured 0.29 -> 0.10, still falling
    w = out["ew"][1]
    step = np.diff(w[5:])                              # W^2 = a + b ln t: equal increments per octave
    assert np.all(step > 0) and step.max() / step.min() < 1.5, step


def test_streamed_kernel_on_a_lattice_beyond_every_on_chip_variant(K):
    """8192 x 8192 (8 MiB of slope planes: no cluster holds it) runs on K5, one launch per colour pass, as the 2^30-site
    bench workload `2d-32768` does.  No oracle run is feasible (30 s per MCS), so: every row and column still closes
    periodically, the surface has moved, and the row-wise exact sums equal a torch reduction of the column-wise heights."""
    L = 8192
    g = K.Kpz2dSim(L, L, 1, 0.75, 0.0, seed=8, max_records=2)
    assert g.path == K.KPZ_PATH_STREAM
    g.set_record_times([3, 6])
    g.run(6)
    r = g.roughness()
    h = g.heights(0).to(torch.int64)
    assert int(h.sum()) == r["sum_h"][1, 0] and int((h * h).sum()) == r["sum_h2"][1, 0]
    assert 0.3 < r["w2_mean"][0] < r["w2_mean"][1] < 1.5
    h = h.view(L, L)
    assert torch.all((h[:, 1:] - h[:, :-1]).abs() == 1) and torch.all((h[1:, :] - h[:-1, :]).abs() == 1)
    assert torch.all((h[:, 0] - h[:, -1]).abs() == 1) and torch.all((h[0, :] - h[-1, :]).abs() == 1)   # periodic closure
