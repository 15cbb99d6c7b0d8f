"""Thin Python binding of libkpz_b200.so (include/kpz_b200.h).

Argument marshalling only: every step of the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for
device memory (workspace and output tensors) and for the CUDA stream — nothing else.  There is no CPU fallback:
a missing library or a missing GPU raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libkpz_b200.so")
HOOKS_PATH = os.path.join(HERE, "libkpz_b200_testhooks.so")

KPZ_PATH_AUTO, KPZ_PATH_ONCHIP, KPZ_PATH_STREAM, KPZ_PATH_BLOCKED = 0, 1, 2, 3
KPZ2D_PATH_CLUSTER = 3     # kpz2d_* only: a sample on chip, spread over a thread-block cluster


class KpzError(RuntimeError):
    def __init__(self, code, what, detail):
        super().__init__(f"{what}: error {code} ({detail})")
        self.code = code


class Disorder(C.Structure):
    _fields_ = [("prob_slow_p", C.c_double), ("p_slow", C.c_double), ("prob_slow_q", C.c_double),
                ("q_slow", C.c_double)]


class Crossing(C.Structure):
    _fields_ = [("prob_flag", C.c_double), ("w_flagged", C.c_double), ("w_unflagged", C.c_double),
                ("independent", C.c_int32)]


class Options(C.Structure):
    _fields_ = [("first_sample", C.c_int32), ("offset_mode", C.c_int32), ("path", C.c_int32)]


_lib = None

# name -> (restype, argtypes); every symbol include/kpz_b200.h declares
_P = C.c_void_p
SIGNATURES = {
    "kpz_workspace_bytes": (C.c_int, [C.c_int64, C.c_int32, C.POINTER(Disorder), C.POINTER(Options), C.c_int32,
                                      C.POINTER(C.c_size_t)]),
    "kpz_create": (C.c_int, [C.POINTER(_P), C.c_int64, C.c_int32, C.c_double, C.c_double, C.POINTER(Disorder),
                             C.c_uint64, C.POINTER(Options), C.c_int32, _P, C.c_size_t, _P]),
    "kpz_set_record_times": (C.c_int, [_P, C.POINTER(C.c_int64), C.c_int32]),
    "kpz_run": (C.c_int, [_P, C.c_int64]),
    "kpz_time": (C.c_int, [_P, C.POINTER(C.c_int64)]),
    "kpz_set_time": (C.c_int, [_P, C.c_int64]),
    "kpz_reset": (C.c_int, [_P]),
    "kpz_lattice": (C.c_int, [_P, _P]),
    "kpz_set_lattice": (C.c_int, [_P, _P]),
    "kpz_disorder_masks": (C.c_int, [_P, _P, _P]),
    "kpz_set_disorder_masks": (C.c_int, [_P, _P, _P]),
    "kpz_heights": (C.c_int, [_P, C.c_int32, _P]),
    "kpz_roughness": (C.c_int, [_P, C.POINTER(C.c_int32), _P, _P, _P, _P]),
    "kpz_destroy": (C.c_int, [_P]),
    "kpz_noalloc_height_sums": (C.c_int, [_P, C.c_int64, C.c_int32, _P, _P, _P]),
    "lanes_workspace_bytes": (C.c_int, [C.c_int64, C.c_int32, C.c_int32, C.POINTER(C.c_size_t)]),
    "lanes_create": (C.c_int, [C.POINTER(_P), C.c_int64, C.c_int32, C.c_double, C.c_double, C.c_double, C.c_double,
                               C.c_int64, C.c_double, C.c_uint64, C.POINTER(Options), C.c_int32, _P, C.c_size_t, _P]),
    "lanes_create_crossing": (C.c_int, [C.POINTER(_P), C.c_int64, C.c_int32, C.c_double, C.c_double, C.c_double,
                                        C.POINTER(Crossing), C.c_int64, C.c_uint64, C.POINTER(Options), C.c_int32, _P,
                                        C.c_size_t, _P]),
    "lanes_flags": (C.c_int, [_P, _P, _P]),
    "lanes_set_flags": (C.c_int, [_P, _P, _P]),
    "lanes_crossing_jit_check": (C.c_int, [C.c_int64, C.c_double, C.c_double, C.POINTER(Crossing), C.c_int64,
                                           C.POINTER(Options), C.POINTER(C.c_size_t)]),
    "lanes_set_record_times": (C.c_int, [_P, C.POINTER(C.c_int64), C.c_int32]),
    "lanes_run": (C.c_int, [_P, C.c_int64]),
    "lanes_time": (C.c_int, [_P, C.POINTER(C.c_int64)]),
    "lanes_set_time": (C.c_int, [_P, C.c_int64]),
    "lanes_reset": (C.c_int, [_P]),
    "lanes_state": (C.c_int, [_P, _P, _P, _P]),
    "lanes_set_state": (C.c_int, [_P, _P, _P, _P]),
    "lanes_currents": (C.c_int, [_P, C.POINTER(C.c_int32), _P, _P, _P, _P, _P]),
    "lanes_profile": (C.c_int, [_P, _P, _P, C.POINTER(C.c_int64)]),
    "lanes_destroy": (C.c_int, [_P]),
    "kpz2d_workspace_bytes": (C.c_int, [C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_size_t)]),
    "kpz2d_create": (C.c_int, [C.POINTER(_P), C.c_int32, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_uint64,
                               C.POINTER(Options), C.c_int32, _P, C.c_size_t, _P]),
    "kpz2d_set_record_times": (C.c_int, [_P, C.POINTER(C.c_int64), C.c_int32]),
    "kpz2d_run": (C.c_int, [_P, C.c_int64]),
    "kpz2d_time": (C.c_int, [_P, C.POINTER(C.c_int64)]),
    "kpz2d_path": (C.c_int, [_P, C.POINTER(C.c_int32)]),
    "kpz2d_reset": (C.c_int, [_P]),
    "kpz2d_slopes": (C.c_int, [_P, _P, _P]),
    "kpz2d_set_slopes": (C.c_int, [_P, _P, _P]),
    "kpz2d_heights": (C.c_int, [_P, C.c_int32, _P]),
    "kpz2d_roughness": (C.c_int, [_P, C.POINTER(C.c_int32), _P, _P, _P, _P]),
    "kpz2d_destroy": (C.c_int, [_P]),
    "kpz_strerror": (C.c_char_p, [C.c_int]),
    "kpz_last_error": (C.c_char_p, []),
    "kpz_kernel_launches": (C.c_int64, []),
    "kpz_path": (C.c_int, [_P, C.POINTER(C.c_int32)]),
    "kpz_debug_config": (C.c_int, [C.c_char_p]),
    "kpz_debug_dump_cubins": (C.c_int, [C.c_char_p, C.POINTER(C.c_int32)]),
    "kpz_jit_check": (C.c_int, [C.c_int64, C.c_double, C.c_double, C.POINTER(Disorder), C.POINTER(Options),
                                C.POINTER(C.c_size_t)]),
    "kpz2d_jit_check": (C.c_int, [C.c_int32, C.c_int32, C.c_double, C.c_double, C.POINTER(Options), C.POINTER(C.c_size_t)]),
    "lanes_jit_check": (C.c_int, [C.c_int64, C.c_double, C.c_double, C.c_double, C.c_int64, C.c_double,
                                  C.POINTER(Options), C.POINTER(C.c_size_t)]),
}


def load_library():
    """Load libkpz_b200.so (built in-tree by paper_1012_0385_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1012_0385_b200.build` "
                "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _chk(rc, what):
    if rc != 0:
        lib = load_library()
        raise KpzError(rc, what, (lib.kpz_last_error() or b"").decode())


def _require_cuda():
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1012_0385_b200 needs a CUDA device (no CPU fallback)")


def _stream_ptr():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _times(t):
    return np.ascontiguousarray(np.asarray(list(t), dtype=np.int64))


def kernel_launches() -> int:
    return int(load_library().kpz_kernel_launches())


class debug_config:
    """kpz_debug_config: test / tuning hook ("jit=0", "K1J_VARIANT=2;K1J_EAGER=3", ...).  Usable as a plain call or as a
    context manager that restores the defaults on exit."""

    def __init__(self, spec: str | None = None):
        _chk(load_library().kpz_debug_config((spec or "").encode()), "kpz_debug_config")

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        _chk(load_library().kpz_debug_config(b""), "kpz_debug_config")
        return False


def debug_dump_cubins(directory: str) -> int:
    """kpz_debug_dump_cubins: every kernel image compiled by this process so far -> <directory>/<entry>_<n>.cubin."""
    os.makedirs(directory, exist_ok=True)
    n = C.c_int32(0)
    _chk(load_library().kpz_debug_dump_cubins(directory.encode(), C.byref(n)), "kpz_debug_dump_cubins")
    return int(n.value)


KPZ_NOALLOC_MAX_TILES = 65536


def noalloc_height_sums(words, L, sum_h, sum_h2) -> None:
    """kpz_noalloc_height_sums: sum h, sum h^2 of the rings in `words` ([nsamples, L/32] int32 / uint32 CUDA tensor, natural
    layout) into the caller's int64 CUDA tensors `sum_h`, `sum_h2` ([nsamples]).  Allocates nothing, on either side of
    the ABI: the scratch is a static device array (nsamples * ceil(L / 65536) <= KPZ_NOALLOC_MAX_TILES).  Asynchronous on
    the current stream; calls that overlap on the GPU race on that array."""
    L = int(L)
    if not (words.is_cuda and sum_h.is_cuda and sum_h2.is_cuda and words.is_contiguous() and sum_h.is_contiguous()
            and sum_h2.is_contiguous()):
        raise ValueError("words, sum_h, sum_h2 must be contiguous CUDA tensors")
    if words.element_size() != 4 or sum_h.dtype != torch.int64 or sum_h2.dtype != torch.int64:
        raise ValueError("words must hold 32-bit words, sum_h / sum_h2 int64")
    if L < 32 or words.numel() % (L // 32) != 0:
        raise ValueError("words must hold nsamples * L/32 words")
    S = words.numel() // (L // 32)
    if sum_h.numel() != S or sum_h2.numel() != S:
        raise ValueError("sum_h, sum_h2 must hold one value per sample")
    with torch.cuda.device(words.device):
        _chk(load_library().kpz_noalloc_height_sums(_dptr(words), L, S, _dptr(sum_h), _dptr(sum_h2), _stream_ptr()),
             "kpz_noalloc_height_sums")


def jit_check(L, p, q, disorder=None, offset_mode=0, path=KPZ_PATH_AUTO) -> int:
    """kpz_jit_check: compile (no GPU needed) the specialised sweep kernel for these parameters; cubin size in bytes."""
    d = None if disorder is None else Disorder(*[float(x) for x in disorder])
    o = Options(0, int(offset_mode), int(path))
    n = C.c_size_t()
    _chk(load_library().kpz_jit_check(int(L), float(p), float(q), C.byref(d) if d is not None else None, C.byref(o),
                                      C.byref(n)), "kpz_jit_check")
    return int(n.value)


def kpz2d_jit_check(Lx, Ly, p, q, offset_mode=0, path=KPZ_PATH_AUTO) -> int:
    """kpz2d_jit_check: compile (no GPU needed) the specialised 2+1D kernel for these parameters; cubin size in bytes."""
    o = Options(0, int(offset_mode), int(path))
    n = C.c_size_t()
    _chk(load_library().kpz2d_jit_check(int(Lx), int(Ly), float(p), float(q), C.byref(o), C.byref(n)), "kpz2d_jit_check")
    return int(n.value)


def lanes_jit_check(L, p_a, p_b, turn_prob, turn_period, omega, offset_mode=0) -> int:
    """lanes_jit_check: compile (no GPU needed) the specialised two-lane kernel; cubin size in bytes."""
    o = Options(0, int(offset_mode), 0)
    n = C.c_size_t()
    _chk(load_library().lanes_jit_check(int(L), float(p_a), float(p_b), float(turn_prob), int(turn_period),
                                        float(omega), C.byref(o), C.byref(n)), "lanes_jit_check")
    return int(n.value)


def lanes_crossing_jit_check(L, p_a, p_b, prob_flag, w_flagged, w_unflagged, independent, turn_period,
                             offset_mode=0) -> int:
    """lanes_crossing_jit_check: compile (no GPU needed) the two-lane kernel of the site-wise crossing model."""
    o = Options(0, int(offset_mode), 0)
    c = Crossing(float(prob_flag), float(w_flagged), float(w_unflagged), int(independent))
    n = C.c_size_t()
    _chk(load_library().lanes_crossing_jit_check(int(L), float(p_a), float(p_b), C.byref(c), int(turn_period),
                                                 C.byref(o), C.byref(n)), "lanes_crossing_jit_check")
    return int(n.value)


class KpzSim:
    """kpz_create / kpz_run / kpz_heights / kpz_roughness on the current CUDA device and stream."""

    def __init__(self, L, nsamples, p, q, disorder=None, seed=0, first_sample=0, offset_mode=0, path=KPZ_PATH_AUTO,
                 max_records=64, device=None):
        _require_cuda()
        lib = load_library()
        self.L, self.S = int(L), int(nsamples)
        self.nw = self.L // 32
        self.device = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
        self._d = None if disorder is None else Disorder(*[float(x) for x in disorder])
        self._o = Options(int(first_sample), int(offset_mode), int(path))
        self.max_records = int(max_records)
        nbytes = C.c_size_t()
        dref = C.byref(self._d) if self._d is not None else None
        _chk(lib.kpz_workspace_bytes(self.L, self.S, dref, C.byref(self._o), self.max_records, C.byref(nbytes)),
             "kpz_workspace_bytes")
        self.workspace = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self._h = C.c_void_p()
        _chk(lib.kpz_create(C.byref(self._h), self.L, self.S, float(p), float(q), dref, int(seed), C.byref(self._o),
                            self.max_records, C.c_void_p(base), nbytes.value, _stream_ptr()), "kpz_create")
        self._nt = 0

    def close(self):
        if getattr(self, "_h", None):
            load_library().kpz_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def path(self):
        p = C.c_int32()
        _chk(load_library().kpz_path(self._h, C.byref(p)), "kpz_path")
        return int(p.value)

    @property
    def time(self):
        t = C.c_int64()
        _chk(load_library().kpz_time(self._h, C.byref(t)), "kpz_time")
        return int(t.value)

    def set_time(self, t):
        """Checkpoint restore: continue from MCS count t (drops the record list)."""
        _chk(load_library().kpz_set_time(self._h, int(t)), "kpz_set_time")
        self._nt = 0

    def set_record_times(self, t):
        t = _times(t)
        self._nt = len(t)
        _chk(load_library().kpz_set_record_times(self._h, t.ctypes.data_as(C.POINTER(C.c_int64)), len(t)),
             "kpz_set_record_times")

    def run(self, n_mcs):
        _chk(load_library().kpz_run(self._h, int(n_mcs)), "kpz_run")

    def reset(self):
        _chk(load_library().kpz_reset(self._h), "kpz_reset")

    def lattice(self, out=None):
        """Occupation words [S][L/32] (natural layout) as a device tensor (int32 storage of the uint32 words)."""
        if out is None:
            out = torch.empty((self.S, self.nw), dtype=torch.int32, device=self.device)
        _chk(load_library().kpz_lattice(self._h, _dptr(out)), "kpz_lattice")
        return out

    def set_lattice(self, words):
        assert words.is_cuda and words.is_contiguous() and words.numel() == self.S * self.nw
        _chk(load_library().kpz_set_lattice(self._h, _dptr(words)), "kpz_set_lattice")

    def disorder_masks(self):
        sp = torch.empty((self.S, self.nw), dtype=torch.int32, device=self.device)
        sq = torch.empty((self.S, self.nw), dtype=torch.int32, device=self.device)
        _chk(load_library().kpz_disorder_masks(self._h, _dptr(sp), _dptr(sq)), "kpz_disorder_masks")
        return sp, sq

    def set_disorder_masks(self, slow_p=None, slow_q=None):
        _chk(load_library().kpz_set_disorder_masks(self._h, _dptr(slow_p), _dptr(slow_q)), "kpz_set_disorder_masks")

    def heights(self, sample, out=None):
        if out is None:
            out = torch.empty(self.L, dtype=torch.int32, device=self.device)
        _chk(load_library().kpz_heights(self._h, int(sample), _dptr(out)), "kpz_heights")
        return out

    def roughness(self):
        """Records so far: dict(t[nt], sum_h[nt][S], sum_h2[nt][S], w2_mean[nt]) as numpy arrays (syncs)."""
        cap = max(self._nt, 1)
        nt = C.c_int32(cap)
        t = np.zeros(cap, dtype=np.int64)
        s1 = np.zeros((cap, self.S), dtype=np.int64)
        s2 = np.zeros((cap, self.S), dtype=np.int64)
        w2 = np.zeros(cap, dtype=np.float64)
        _chk(load_library().kpz_roughness(self._h, C.byref(nt), t.ctypes.data, s1.ctypes.data, s2.ctypes.data,
                                          w2.ctypes.data), "kpz_roughness")
        k = nt.value
        return dict(t=t[:k], sum_h=s1[:k], sum_h2=s2[:k], w2_mean=w2[:k])


class Kpz2dSim:
    """kpz2d_create / kpz2d_run / kpz2d_heights / kpz2d_roughness (the 2+1D generalisation) on the current
    CUDA device and stream.  Argument marshalling only."""

    def __init__(self, Lx, Ly, nsamples, p, q, seed=0, first_sample=0, offset_mode=0, max_records=64, path=KPZ_PATH_AUTO):
        _require_cuda()
        lib = load_library()
        self.Lx, self.Ly, self.S = int(Lx), int(Ly), int(nsamples)
        self.rw = self.Lx // 32
        self.max_records = int(max_records)
        self.device = torch.device("cuda", torch.cuda.current_device())
        self._o = Options(int(first_sample), int(offset_mode), int(path))
        nbytes = C.c_size_t()
        _chk(lib.kpz2d_workspace_bytes(self.Lx, self.Ly, self.S, self.max_records, C.byref(nbytes)), "kpz2d_workspace_bytes")
        self.workspace = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self._h = C.c_void_p()
        _chk(lib.kpz2d_create(C.byref(self._h), self.Lx, self.Ly, self.S, float(p), float(q), int(seed), C.byref(self._o),
                              self.max_records, C.c_void_p(base), nbytes.value, _stream_ptr()), "kpz2d_create")
        self._nt = 0

    def close(self):
        if getattr(self, "_h", None):
            load_library().kpz2d_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def path(self):
        p = C.c_int32()
        _chk(load_library().kpz2d_path(self._h, C.byref(p)), "kpz2d_path")
        return int(p.value)

    @property
    def time(self):
        t = C.c_int64()
        _chk(load_library().kpz2d_time(self._h, C.byref(t)), "kpz2d_time")
        return int(t.value)

    def set_record_times(self, t):
        t = _times(t)
        self._nt = len(t)
        _chk(load_library().kpz2d_set_record_times(self._h, t.ctypes.data_as(C.POINTER(C.c_int64)), len(t)),
             "kpz2d_set_record_times")

    def run(self, n_mcs):
        _chk(load_library().kpz2d_run(self._h, int(n_mcs)), "kpz2d_run")

    def reset(self):
        _chk(load_library().kpz2d_reset(self._h), "kpz2d_reset")

    def slopes(self):
        """(sx, sy): device tensors [S][Ly][Lx/32] (int32 storage of the uint32 words)."""
        sx = torch.empty((self.S, self.Ly, self.rw), dtype=torch.int32, device=self.device)
        sy = torch.empty_like(sx)
        _chk(load_library().kpz2d_slopes(self._h, _dptr(sx), _dptr(sy)), "kpz2d_slopes")
        return sx, sy

    def set_slopes(self, sx, sy):
        assert sx.is_cuda and sx.is_contiguous() and sx.numel() == self.S * self.Ly * self.rw and sy.numel() == sx.numel()
        _chk(load_library().kpz2d_set_slopes(self._h, _dptr(sx), _dptr(sy)), "kpz2d_set_slopes")

    def heights(self, sample):
        out = torch.empty((self.Ly, self.Lx), dtype=torch.int32, device=self.device)
        _chk(load_library().kpz2d_heights(self._h, int(sample), _dptr(out)), "kpz2d_heights")
        return out

    def roughness(self):
        cap = max(self._nt, 1)
        nt = C.c_int32(cap)
        t = np.zeros(cap, dtype=np.int64)
        s1 = np.zeros((cap, self.S), dtype=np.int64)
        s2 = np.zeros((cap, self.S), dtype=np.int64)
        w2 = np.zeros(cap, dtype=np.float64)
        _chk(load_library().kpz2d_roughness(self._h, C.byref(nt), t.ctypes.data, s1.ctypes.data, s2.ctypes.data,
                                            w2.ctypes.data), "kpz2d_roughness")
        k = nt.value
        return dict(t=t[:k], sum_h=s1[:k], sum_h2=s2[:k], w2_mean=w2[:k])


class LanesSim:
    """lanes_create / lanes_run / lanes_currents / lanes_profile on the current CUDA device and stream."""

    def __init__(self, L, nsamples, p_a, p_b, rho0, turn_prob, turn_period, omega, seed=0, first_sample=0,
                 offset_mode=0, max_records=64, device=None, w_unflagged=None, independent=0):
        """w_unflagged=None: lanes_create (turning-point model); otherwise lanes_create_crossing with
        {prob_flag=turn_prob, w_flagged=omega, w_unflagged, independent} (the paper's own model)."""
        _require_cuda()
        lib = load_library()
        self.L, self.S = int(L), int(nsamples)
        self.nw = self.L // 32
        self.device = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
        self._o = Options(int(first_sample), int(offset_mode), 0)
        self.max_records = int(max_records)
        nbytes = C.c_size_t()
        _chk(lib.lanes_workspace_bytes(self.L, self.S, self.max_records, C.byref(nbytes)), "lanes_workspace_bytes")
        self.workspace = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self._h = C.c_void_p()
        if w_unflagged is None:
            _chk(lib.lanes_create(C.byref(self._h), self.L, self.S, float(p_a), float(p_b), float(rho0),
                                  float(turn_prob), int(turn_period), float(omega), int(seed), C.byref(self._o),
                                  self.max_records, C.c_void_p(base), nbytes.value, _stream_ptr()), "lanes_create")
        else:
            c = Crossing(float(turn_prob), float(omega), float(w_unflagged), int(independent))
            _chk(lib.lanes_create_crossing(C.byref(self._h), self.L, self.S, float(p_a), float(p_b), float(rho0),
                                           C.byref(c), int(turn_period), int(seed), C.byref(self._o),
                                           self.max_records, C.c_void_p(base), nbytes.value, _stream_ptr()),
                 "lanes_create_crossing")
        self._nt = 0

    def flags(self):
        u, v = [torch.empty((self.S, self.nw), dtype=torch.int32, device=self.device) for _ in range(2)]
        _chk(load_library().lanes_flags(self._h, _dptr(u), _dptr(v)), "lanes_flags")
        return u, v

    def set_flags(self, u=None, v=None):
        _chk(load_library().lanes_set_flags(self._h, _dptr(u), _dptr(v)), "lanes_set_flags")

    def close(self):
        if getattr(self, "_h", None):
            load_library().lanes_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def time(self):
        t = C.c_int64()
        _chk(load_library().lanes_time(self._h, C.byref(t)), "lanes_time")
        return int(t.value)

    def set_time(self, t):
        """Checkpoint restore: continue from MCS count t (drops the record list)."""
        _chk(load_library().lanes_set_time(self._h, int(t)), "lanes_set_time")
        self._nt = 0

    def set_record_times(self, t):
        t = _times(t)
        self._nt = len(t)
        _chk(load_library().lanes_set_record_times(self._h, t.ctypes.data_as(C.POINTER(C.c_int64)), len(t)),
             "lanes_set_record_times")

    def run(self, n_mcs):
        _chk(load_library().lanes_run(self._h, int(n_mcs)), "lanes_run")

    def reset(self):
        _chk(load_library().lanes_reset(self._h), "lanes_reset")

    def state(self):
        a, b, tn = [torch.empty((self.S, self.nw), dtype=torch.int32, device=self.device) for _ in range(3)]
        _chk(load_library().lanes_state(self._h, _dptr(a), _dptr(b), _dptr(tn)), "lanes_state")
        return a, b, tn

    def set_state(self, a=None, b=None, turn=None):
        _chk(load_library().lanes_set_state(self._h, _dptr(a), _dptr(b), _dptr(turn)), "lanes_set_state")

    def currents(self):
        cap = max(self._nt, 1)
        nt = C.c_int32(cap)
        t = np.zeros(cap, dtype=np.int64)
        arrs = [np.zeros((cap, self.S), dtype=np.int64) for _ in range(4)]
        _chk(load_library().lanes_currents(self._h, C.byref(nt), t.ctypes.data, *[a.ctypes.data for a in arrs]),
             "lanes_currents")
        k = nt.value
        return dict(t=t[:k], j_a=arrs[0][:k], j_b=arrs[1][:k], n_a=arrs[2][:k], n_b=arrs[3][:k])

    def profile(self):
        oa = torch.empty((self.S, self.L), dtype=torch.int32, device=self.device)
        ob = torch.empty((self.S, self.L), dtype=torch.int32, device=self.device)
        ns = C.c_int64()
        _chk(load_library().lanes_profile(self._h, _dptr(oa), _dptr(ob), C.byref(ns)), "lanes_profile")
        return oa, ob, int(ns.value)


def words_to_numpy(t: torch.Tensor) -> np.ndarray:
    """Device int32 word tensor -> host uint32 numpy array (marshalling only)."""
    return t.detach().cpu().numpy().view(np.uint32)


def words_from_numpy(a: np.ndarray, device) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint32).view(np.int32)).to(device)
