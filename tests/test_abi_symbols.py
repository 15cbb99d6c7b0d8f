"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol include/kpz_b200.h declares
(no compute calls here).  Argument validation that needs no device is checked too."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1012_0385_b200 import build
    build.build()
    from paper_1012_0385_b200 import binding
    return binding.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "kpz_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b((?:kpz2d|kpz|lanes)_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_all_exported_and_bound(lib):
    from paper_1012_0385_b200 import binding
    names = _declared_symbols()
    assert len(names) >= 26
    for n in names:
        assert hasattr(lib, n), n
        assert n in binding.SIGNATURES, f"{n} has no ctypes signature in the binding"
    assert sorted(binding.SIGNATURES) == names


def test_sizes_and_argument_validation_without_a_device(lib):
    from paper_1012_0385_b200.binding import Disorder, Options
    n = C.c_size_t()
    assert lib.kpz_workspace_bytes(8192, 1024, None, None, 40, C.byref(n)) == 0
    assert n.value >= 1024 * 8192 // 8
    small = n.value
    d = Disorder(0.1, 0.5, 0.0, 0.0)
    assert lib.kpz_workspace_bytes(8192, 1024, C.byref(d), None, 40, C.byref(n)) == 0
    assert n.value > small
    # streamed path: ping-pong buffers
    o = Options(0, 0, 2)
    assert lib.kpz_workspace_bytes(1 << 28, 1, None, C.byref(o), 20, C.byref(n)) == 0
    assert n.value >= 2 * (1 << 28) // 8
    # errors: L not a multiple of 64 -> EUNSUPPORTED (-2); odd L -> EINVAL (-1); forced on-chip too large -> -2
    assert lib.kpz_workspace_bytes(100, 1, None, None, 1, C.byref(n)) == -2
    assert b"multiple of 64" in lib.kpz_last_error()
    assert lib.kpz_workspace_bytes(63, 1, None, None, 1, C.byref(n)) == -1
    o1 = Options(0, 0, 1)
    assert lib.kpz_workspace_bytes(1 << 20, 1, None, C.byref(o1), 1, C.byref(n)) == -2
    assert lib.kpz_workspace_bytes(64, 0, None, None, 1, C.byref(n)) == -1
    assert lib.lanes_workspace_bytes(16384, 256, 50, C.byref(n)) == 0
    assert n.value >= 2 * 256 * 16384 * 4
    assert lib.lanes_workspace_bytes(1 << 20, 1, 1, C.byref(n)) == -2
    h = C.c_void_p()
    assert lib.kpz_create(C.byref(h), 64, 1, 1.5, 0.0, None, 1, None, 1, None, 0, None) == -1   # p outside [0,1]
    assert lib.kpz_create(C.byref(h), 64, 1, 0.5, 0.0, None, 1, None, 1, None, 0, None) == -1   # NULL workspace
    assert lib.kpz_strerror(-4) == b"CUDA error" and lib.kpz_strerror(0) == b"ok"
    assert lib.kpz_kernel_launches() == 0


def test_binding_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    from paper_1012_0385_b200 import KpzSim
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        KpzSim(64, 1, 0.5, 0.5)
