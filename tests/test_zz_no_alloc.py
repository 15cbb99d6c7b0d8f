"""kpz_noalloc_height_sums: the allocation-free entry point (static device scratch) against the existing paths.

Collected last on purpose (the suite runs with `pytest -x`; a failure here hides nothing).  The entry point shares one
static scratch array between all calls, so the cases run back to back in ONE test: several tiles per ring first (which
leaves tile bases behind), then one tile per ring (which needs them cleared), then a rough lattice; every call's
outputs are pre-filled with garbage.  Integer work: the comparison is bit-exact, as in the other GPU tests.

Existing paths compared against:
  * the fused reduction of kpz_run at a record time (kpz_roughness) for the lattice kpz_lattice returns at that time;
  * kpz_heights (int32 heights of a lattice handed in with kpz_set_lattice) summed by torch in int64.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def K():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1012_0385_b200 as pkg
    pkg.load_library()
    return pkg


def _evolved(K, L, S, n_mcs, seed, p=0.75, q=0.25):
    """Rings after n_mcs MCS and the sums the existing fused reduction captured at that time."""
    sim = K.KpzSim(L, S, p, q, seed=seed, max_records=1)
    sim.set_record_times([n_mcs])
    sim.run(n_mcs)
    lat = sim.lattice()
    r = sim.roughness()
    assert list(r["t"]) == [n_mcs]
    sim.close()
    return lat, r["sum_h"][0], r["sum_h2"][0]


def _call(K, lat, L):
    S = lat.numel() // (L // 32)
    out_h = torch.full((S,), 0x5A5A5A5A5A5A, dtype=torch.int64, device=lat.device)    # garbage: the call must overwrite
    out_h2 = torch.full((S,), -77, dtype=torch.int64, device=lat.device)
    K.noalloc_height_sums(lat, L, out_h, out_h2)
    return out_h.cpu().numpy(), out_h2.cpu().numpy()


def test_noalloc_height_sums_two_calls_in_a_row_match_the_existing_paths(K):
    # call 1: 3 rings of 2^20 sites = 16 tiles each (streamed path of the library), tile bases left in the scratch
    L1 = 1 << 20
    lat1, h1, h2_1 = _evolved(K, L1, 3, 24, seed=5)
    a, b = _call(K, lat1, L1)
    assert np.array_equal(a, h1) and np.array_equal(b, h2_1)
    assert np.all(b > 0) and not np.array_equal(b, np.full(3, L1))          # not the flat start's sums

    # call 2, right after: 50 ragged one-warp rings (L = 64 * 37), ONE tile per ring - stale tile bases would be added
    L2 = 64 * 37
    lat2, h, h2 = _evolved(K, L2, 50, 200, seed=6, p=0.9, q=0.1)
    a, b = _call(K, lat2, L2)
    assert np.array_equal(a, h) and np.array_equal(b, h2)

    # call 3: the same inputs again -> the same outputs (nothing accumulates between calls)
    a2, b2 = _call(K, lat2, L2)
    assert np.array_equal(a2, a) and np.array_equal(b2, b)

    # call 4: call 1's rings again, after the small calls overwrote the head of the scratch
    a, b = _call(K, lat1, L1)
    assert np.array_equal(a, h1) and np.array_equal(b, h2_1)

    # call 5: rough rings (random occupation, particle number != L/2), a ragged second tile: L = 64 * 1031 = 65984 sites;
    # existing path = kpz_set_lattice + kpz_heights, summed by torch
    L3, S3 = 64 * 1031, 5
    g = torch.Generator(device="cpu").manual_seed(11)
    words = torch.randint(-2**31, 2**31, (S3, L3 // 32), generator=g, dtype=torch.int64).to(torch.int32).cuda()
    sim = K.KpzSim(L3, S3, 0.5, 0.5, seed=1, max_records=1)
    sim.set_lattice(words)
    exp_h, exp_h2 = [], []
    for s in range(S3):
        hh = sim.heights(s).to(torch.int64)
        exp_h.append(int(hh.sum()))
        exp_h2.append(int((hh * hh).sum()))
    sim.close()
    a, b = _call(K, words, L3)
    assert list(a) == exp_h and list(b) == exp_h2


def test_noalloc_call_does_not_move_free_device_memory(K):
    L, S = 1 << 17, 4
    lat, h, h2 = _evolved(K, L, S, 8, seed=9)
    out_h = torch.empty(S, dtype=torch.int64, device="cuda")
    out_h2 = torch.empty(S, dtype=torch.int64, device="cuda")
    K.noalloc_height_sums(lat, L, out_h, out_h2)          # first use may load the kernels' module
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        K.noalloc_height_sums(lat, L, out_h, out_h2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert np.array_equal(out_h.cpu().numpy(), h) and np.array_equal(out_h2.cpu().numpy(), h2)


def test_noalloc_rejects_sizes_beyond_its_static_scratch(K):
    dummy = torch.zeros(64, dtype=torch.int32, device="cuda")
    out = torch.zeros(1, dtype=torch.int64, device="cuda")
    lib = K.load_library()
    import ctypes as C
    def raw(L, S):
        return lib.kpz_noalloc_height_sums(C.c_void_p(dummy.data_ptr()), L, S, C.c_void_p(out.data_ptr()),
                                           C.c_void_p(out.data_ptr()), None)
    # sizes are checked before any pointer is used, so the small dummy buffers are never touched
    assert raw(1 << 20, K.KPZ_NOALLOC_MAX_TILES // 16 + 1) == -2           # one tile too many
    assert b"KPZ_NOALLOC_MAX_TILES" in lib.kpz_last_error()
    assert raw((1 << 30) + 64, 1) == -2                                    # ring too long
    assert raw(64 * 3 + 32, 1) == -2                                       # not a multiple of 64
    assert raw(32, 1) == -1 and raw(64, 0) == -1
    assert lib.kpz_noalloc_height_sums(None, 64, 1, C.c_void_p(out.data_ptr()), C.c_void_p(out.data_ptr()), None) == -1
    # four times the ensemble of BASELINE config 3 in one call (4096 of the 65536 tiles)
    S = 4096
    lat = torch.full((S, 16384 // 32), -0x55555556, dtype=torch.int32, device="cuda")     # flat start n_i = i & 1
    oh = torch.empty(S, dtype=torch.int64, device="cuda")
    oh2 = torch.empty(S, dtype=torch.int64, device="cuda")
    K.noalloc_height_sums(lat, 16384, oh, oh2)
    assert torch.all(oh == -16384 // 2) and torch.all(oh2 == 16384 // 2)   # h = -1, 0, -1, 0, ...
