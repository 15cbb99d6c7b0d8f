"""The run-time specialised kernels (NVRTC, csrc/jit.cu) compile for sm_100a WITHOUT a GPU for every BASELINE.json
configuration and for the edge shapes of each code path (no compute calls here): the LUT path (<= 3 selection
inputs), the GENERAL path (tags + planes, non-dyadic rates), ragged rings, multi-warp rings, both offset modes, the
streamed pass kernel, the temporally blocked window kernel and the two-lane kernel."""
import pytest

import workloads


@pytest.fixture(scope="module")
def K():
    from paper_1012_0385_b200 import build
    build.build()
    import paper_1012_0385_b200 as pkg
    pkg.load_library()
    return pkg


@pytest.mark.parametrize("key", [1, 2, 3, 4, "4-aux-i"])
def test_kpz_configs_compile(K, key):
    c = workloads.CONFIGS[key]
    n = K.jit_check(c["L"], c["p"], c["q"], disorder=c["disorder"], path=c.get("path", 0))
    assert n > 10_000          # a real sm_100a cubin (per-sample, blocked or pass-by-pass kernel)
    if c.get("path", 0) == K.KPZ_PATH_STREAM:
        with K.debug_config("K1J_PDL=0"):       # the pass kernel without programmatic dependent launch
            assert K.jit_check(c["L"], c["p"], c["q"], disorder=c["disorder"], path=K.KPZ_PATH_STREAM) > 10_000


def test_config5_two_lane_compiles(K):
    c = workloads.CONFIGS[5]
    assert K.lanes_jit_check(c["L"], c["p_a"], c["p_b"], c["turn_prob"], c["turn_period"], c["omega"]) > 10_000


@pytest.mark.parametrize("L,p,q,dis,mode,path", [
    (64, 1.0, 0.0, None, 0, 1),                       # smallest ring, no plane
    (320, 0.5, 0.5, None, 1, 1),                      # ragged unit, alternating offsets, 1 plane
    (8192 + 64, 0.8, 0.0, None, 0, 1),                # 30-plane threshold: GENERAL path with a lazy tail, ragged
    (16384, 0.75, 0.25, (0.5, 0.375, 0.5, 0.125), 0, 1),   # two tag classes + 3 planes: GENERAL, all planes eager
    (1 << 18, 0.75, 0.25, None, 0, 1),                # 1024 threads per ring
    (1 << 18, 0.9, 0.1, (0.1, 0.5, 0.0, 0.0), 0, 3),  # blocked window kernel with tags
    (64, 0.75, 0.25, None, 1, 3),                     # ring shorter than a window
])
def test_edge_shapes_compile(K, L, p, q, dis, mode, path):
    assert K.jit_check(L, p, q, disorder=dis, offset_mode=mode, path=path) > 10_000


@pytest.mark.parametrize("L,pa,pb,turn,period,omega", [
    (64, 1.0, 1.0, 0.05, 100, 0.1),
    (64 * 5, 0.75, 0.5, 0.25, 0, 0.5),      # ragged, in-lane planes, turning points never redrawn
    (131072, 1.0, 0.75, 0.05, 7, 1.0),      # largest ring of the specialised kernel
])
def test_two_lane_edge_shapes_compile(K, L, pa, pb, turn, period, omega):
    assert K.lanes_jit_check(L, pa, pb, turn, period, omega) > 10_000


@pytest.mark.parametrize("L,indep,period", [(512, 1, 0), (4096, 1, 100), (131072, 0, 0)])
def test_paper_two_lane_model_compiles(K, L, indep, period):
    assert K.lanes_crossing_jit_check(L, 0.5, 0.5, 0.5, 0.2, 0.8, indep, period) > 10_000


@pytest.mark.parametrize("Lx,Ly,p,q,path", [
    (512, 512, 0.75, 0.0, 0),       # bench workload 2d-512: on chip, two planes, a row = two lanes of a warp
    (1024, 1024, 0.75, 0.0, 0),     # 2d-1024: streamed
    (512, 512, 0.8, 0.1, 1),        # lazy plane loop on chip
    (64, 16, 0.75, 0.25, 0),        # ragged: a supergroup spans rows
    (320, 10, 0.3, 0.2, 2),
    (256, 2, 1.0, 0.0, 1),          # one supergroup per row, Ly = 2
    (768, 64, 0.5, 0.5, 1),         # three supergroups per row: no shuffles
    (8192, 4, 0.75, 0.0, 1),        # a row longer than a warp
])
def test_2d_kernels_compile(K, Lx, Ly, p, q, path):
    assert K.kpz2d_jit_check(Lx, Ly, p, q, path=path) > 10_000
    with K.debug_config("K5J_RIW=0"):
        assert K.kpz2d_jit_check(Lx, Ly, p, q, path=path) > 10_000
    with K.debug_config("jit=0"):
        assert K.kpz2d_jit_check(Lx, Ly, p, q, path=path) == 0


def test_bad_arguments_are_refused_without_compiling(K):
    with pytest.raises(K.KpzError):
        K.kpz2d_jit_check(100, 64, 0.5, 0.5)    # Lx not a multiple of 64
    with pytest.raises(K.KpzError):
        K.kpz2d_jit_check(2048, 2048, 0.5, 0.5, path=1)   # beyond the shared memory of an SM
    with pytest.raises(K.KpzError):
        K.jit_check(100, 0.5, 0.5)              # L not a multiple of 64
    with pytest.raises(K.KpzError):
        K.jit_check(64, 1.5, 0.5)
    with pytest.raises(K.KpzError):
        K.lanes_jit_check(64, 1.0, 1.0, 0.05, -1, 0.1)


@pytest.mark.parametrize("variant", ["0", "1", "2"])
def test_every_code_shape_of_the_sweep_compiles(K, variant):
    """K1J_VARIANT: 4-way switch with the Philox rounds inside, branch-free, 4-way switch after the Philox rounds."""
    with K.debug_config("K1J_VARIANT=" + variant):
        assert K.jit_check(8192, 0.75, 0.25) > 10_000
        assert K.jit_check(16384, 1.0, 0.0, disorder=(0.1, 0.5, 0.0, 0.0)) > 10_000
        assert K.jit_check(1 << 20, 0.75, 0.25, path=3) > 10_000


def test_debug_config_is_validated_and_restored(K):
    with pytest.raises(K.KpzError):
        K.debug_config("FOO=1")
    with pytest.raises(K.KpzError):
        K.debug_config("K1J_VARIANT")
    with pytest.raises(K.KpzError):
        K.debug_config("K1J_X=1 -DY")
    with K.debug_config("jit=0"):
        assert K.jit_check(8192, 0.75, 0.25) == 0          # statically compiled kernel: nothing to specialise
    assert K.jit_check(8192, 0.75, 0.25) > 10_000


def test_compiled_images_can_be_dumped(K, tmp_path):
    K.jit_check(8192, 0.75, 0.25)
    n = K.debug_dump_cubins(str(tmp_path))
    assert n >= 1
    names = sorted(p.name for p in tmp_path.iterdir())
    assert any(x.startswith("kpz_k1_sweep_jit_") and x.endswith(".cubin") for x in names)
    txts = [p.read_text() for p in tmp_path.iterdir() if p.name.startswith("kpz_k1_sweep_jit_") and p.suffix == ".txt"]
    assert any("-DK1J_PW=128" in t for t in txts)       # L = 8192: 128 words per parity plane
