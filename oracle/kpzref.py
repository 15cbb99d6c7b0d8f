"""ctypes loader for the CPU oracle (oracle/kpz_oracle.c).  TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
Argument marshalling only; every number comes from the C oracle.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None

TAGS = dict(PAIR=0, OFFSET=1, SLOW_P=2, SLOW_Q=3, INIT_A=4, INIT_B=5, PAIR_B=6, TURN=7, SWITCH_AB=8,
            SWITCH_BA=9, RSU=10, TURN_V=11)


class Disorder(C.Structure):
    _fields_ = [("prob_slow_p", C.c_double), ("p_slow", C.c_double), ("prob_slow_q", C.c_double),
                ("q_slow", C.c_double)]


class Options(C.Structure):
    _fields_ = [("first_sample", C.c_int32), ("offset_mode", C.c_int32), ("path", C.c_int32)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.kpzref_philox4x32_10.restype = None
    return _lib


class OracleError(RuntimeError):
    pass


def _chk(rc, what):
    if rc != 0:
        raise OracleError(f"{what} failed with code {rc}")


def _p(a, ty):
    return None if a is None else a.ctypes.data_as(C.POINTER(ty))


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    out = (C.c_uint32 * 4)()
    lib().kpzref_philox4x32_10(c, k, out)
    return [int(x) for x in out]


def philox_call(seed, tag, sample, timekey, pass_, plane, G):
    out = (C.c_uint32 * 4)()
    _chk(lib().kpzref_philox_call(C.c_uint64(seed), C.c_uint32(tag), C.c_uint32(sample), C.c_uint64(timekey),
                                  C.c_uint32(pass_), C.c_uint32(plane), C.c_uint32(G), out), "philox_call")
    return [int(x) for x in out]


def uniform(seed, tag, sample, timekey, pass_, element):
    u = C.c_uint32()
    _chk(lib().kpzref_uniform(C.c_uint64(seed), C.c_uint32(tag), C.c_uint32(sample), C.c_uint64(timekey),
                              C.c_uint32(pass_), C.c_uint64(element), C.byref(u)), "uniform")
    return int(u.value)


def threshold(x):
    T = C.c_uint64()
    _chk(lib().kpzref_threshold(C.c_double(x), C.byref(T)), "threshold")
    return int(T.value)


def offset(seed, sample, mcs, pass_):
    o = C.c_uint32()
    _chk(lib().kpzref_offset(C.c_uint64(seed), C.c_uint32(sample), C.c_uint64(mcs), C.c_uint32(pass_), C.byref(o)),
         "offset")
    return int(o.value)


def _times(t):
    return np.ascontiguousarray(np.asarray(list(t), dtype=np.int64))


class KpzRef:
    """Oracle KPZ/ASEP ring ensemble (host memory)."""

    def __init__(self, L, nsamples, p, q, disorder=None, seed=0, first_sample=0, offset_mode=0):
        self.L, self.S = int(L), int(nsamples)
        self.nw = (self.L + 31) // 32
        self._h = C.c_void_p()
        d = None
        if disorder is not None:
            d = Disorder(*[float(x) for x in disorder])
        o = Options(int(first_sample), int(offset_mode), 0)
        _chk(lib().kpzref_create(C.byref(self._h), C.c_int64(self.L), C.c_int32(self.S), C.c_double(p),
                                 C.c_double(q), C.byref(d) if d is not None else None, C.c_uint64(seed),
                                 C.byref(o)), "kpzref_create")
        self._nt = 0

    def close(self):
        if self._h:
            lib().kpzref_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_record_times(self, t):
        t = _times(t)
        self._nt = len(t)
        _chk(lib().kpzref_set_record_times(self._h, _p(t, C.c_int64), C.c_int32(len(t))), "set_record_times")

    def run(self, n_mcs):
        _chk(lib().kpzref_run(self._h, C.c_int64(n_mcs)), "kpzref_run")

    def run_rsu(self, n_mcs):
        _chk(lib().kpzref_run_rsu(self._h, C.c_int64(n_mcs)), "kpzref_run_rsu")

    @property
    def time(self):
        t = C.c_int64()
        _chk(lib().kpzref_time(self._h, C.byref(t)), "kpzref_time")
        return int(t.value)

    def set_time(self, t):
        _chk(lib().kpzref_set_time(self._h, C.c_int64(t)), "kpzref_set_time")

    def lattice(self):
        w = np.zeros((self.S, self.nw), dtype=np.uint32)
        _chk(lib().kpzref_lattice(self._h, _p(w, C.c_uint32)), "kpzref_lattice")
        return w

    def set_lattice(self, words):
        w = np.ascontiguousarray(words, dtype=np.uint32).reshape(self.S, self.nw)
        _chk(lib().kpzref_set_lattice(self._h, _p(w, C.c_uint32)), "kpzref_set_lattice")

    def sites(self):
        """Occupations as a uint8 array [S][L]."""
        return unpack_words(self.lattice(), self.L)

    def disorder_masks(self):
        sp = np.zeros((self.S, self.nw), dtype=np.uint32)
        sq = np.zeros((self.S, self.nw), dtype=np.uint32)
        _chk(lib().kpzref_disorder_masks(self._h, _p(sp, C.c_uint32), _p(sq, C.c_uint32)), "kpzref_disorder_masks")
        return sp, sq

    def set_disorder_masks(self, slow_p=None, slow_q=None):
        sp = None if slow_p is None else np.ascontiguousarray(slow_p, dtype=np.uint32).reshape(self.S, self.nw)
        sq = None if slow_q is None else np.ascontiguousarray(slow_q, dtype=np.uint32).reshape(self.S, self.nw)
        _chk(lib().kpzref_set_disorder_masks(self._h, _p(sp, C.c_uint32), _p(sq, C.c_uint32)),
             "kpzref_set_disorder_masks")

    def heights(self, sample):
        h = np.zeros(self.L, dtype=np.int32)
        _chk(lib().kpzref_heights(self._h, C.c_int32(sample), _p(h, C.c_int32)), "kpzref_heights")
        return h

    def roughness(self):
        cap = max(self._nt, 1)
        nt = C.c_int32(cap)
        t = np.zeros(cap, dtype=np.int64)
        s1 = np.zeros((cap, self.S), dtype=np.int64)
        s2 = np.zeros((cap, self.S), dtype=np.int64)
        w2 = np.zeros(cap, dtype=np.float64)
        _chk(lib().kpzref_roughness(self._h, C.byref(nt), _p(t, C.c_int64), _p(s1, C.c_int64), _p(s2, C.c_int64),
                                    _p(w2, C.c_double)), "kpzref_roughness")
        k = nt.value
        return dict(t=t[:k], sum_h=s1[:k], sum_h2=s2[:k], w2_mean=w2[:k])

    def hops(self):
        f = np.zeros(self.S, dtype=np.int64)
        b = np.zeros(self.S, dtype=np.int64)
        _chk(lib().kpzref_hops(self._h, _p(f, C.c_int64), _p(b, C.c_int64)), "kpzref_hops")
        return f, b


class LanesRef:
    """Oracle two-lane model ensemble (host memory)."""

    def __init__(self, L, nsamples, p_a, p_b, rho0, turn_prob, turn_period, omega, seed=0, first_sample=0,
                 offset_mode=0, w_unflagged=None, independent=0):
        """w_unflagged=None: the turning-point model (crossing only at flagged sites, one flag set);
        otherwise the paper's model (§R18): crossing probability omega at flagged sites, w_unflagged elsewhere."""
        self.L, self.S = int(L), int(nsamples)
        self.nw = (self.L + 31) // 32
        self._h = C.c_void_p()
        o = Options(int(first_sample), int(offset_mode), 0)
        if w_unflagged is None:
            _chk(lib().lanesref_create(C.byref(self._h), C.c_int64(self.L), C.c_int32(self.S), C.c_double(p_a),
                                       C.c_double(p_b), C.c_double(rho0), C.c_double(turn_prob),
                                       C.c_int64(turn_period), C.c_double(omega), C.c_uint64(seed), C.byref(o)),
                 "lanesref_create")
        else:
            _chk(lib().lanesref_create_crossing(C.byref(self._h), C.c_int64(self.L), C.c_int32(self.S),
                                                C.c_double(p_a), C.c_double(p_b), C.c_double(rho0),
                                                C.c_double(turn_prob), C.c_double(omega), C.c_double(w_unflagged),
                                                C.c_int32(independent), C.c_int64(turn_period), C.c_uint64(seed),
                                                C.byref(o)), "lanesref_create_crossing")
        self._nt = 0

    def flags(self):
        u = np.zeros((self.S, self.nw), dtype=np.uint32)
        v = np.zeros((self.S, self.nw), dtype=np.uint32)
        _chk(lib().lanesref_flags(self._h, _p(u, C.c_uint32), _p(v, C.c_uint32)), "lanesref_flags")
        return u, v

    def set_flags(self, u=None, v=None):
        def prep(x):
            return None if x is None else np.ascontiguousarray(x, dtype=np.uint32).reshape(self.S, self.nw)
        u, v = prep(u), prep(v)
        _chk(lib().lanesref_set_flags(self._h, _p(u, C.c_uint32), _p(v, C.c_uint32)), "lanesref_set_flags")

    def close(self):
        if self._h:
            lib().lanesref_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_record_times(self, t):
        t = _times(t)
        self._nt = len(t)
        _chk(lib().lanesref_set_record_times(self._h, _p(t, C.c_int64), C.c_int32(len(t))), "set_record_times")

    def run(self, n_mcs):
        _chk(lib().lanesref_run(self._h, C.c_int64(n_mcs)), "lanesref_run")

    @property
    def time(self):
        t = C.c_int64()
        _chk(lib().lanesref_time(self._h, C.byref(t)), "lanesref_time")
        return int(t.value)

    def set_time(self, t):
        _chk(lib().lanesref_set_time(self._h, C.c_int64(t)), "lanesref_set_time")

    def state(self):
        a = np.zeros((self.S, self.nw), dtype=np.uint32)
        b = np.zeros((self.S, self.nw), dtype=np.uint32)
        tn = np.zeros((self.S, self.nw), dtype=np.uint32)
        _chk(lib().lanesref_state(self._h, _p(a, C.c_uint32), _p(b, C.c_uint32), _p(tn, C.c_uint32)),
             "lanesref_state")
        return a, b, tn

    def set_state(self, a=None, b=None, turn=None):
        def prep(x):
            return None if x is None else np.ascontiguousarray(x, dtype=np.uint32).reshape(self.S, self.nw)
        a, b, turn = prep(a), prep(b), prep(turn)
        _chk(lib().lanesref_set_state(self._h, _p(a, C.c_uint32), _p(b, C.c_uint32), _p(turn, C.c_uint32)),
             "lanesref_set_state")

    def currents(self):
        cap = max(self._nt, 1)
        nt = C.c_int32(cap)
        t = np.zeros(cap, dtype=np.int64)
        arrs = [np.zeros((cap, self.S), dtype=np.int64) for _ in range(4)]
        _chk(lib().lanesref_currents(self._h, C.byref(nt), _p(t, C.c_int64), *[_p(a, C.c_int64) for a in arrs]),
             "lanesref_currents")
        k = nt.value
        return dict(t=t[:k], j_a=arrs[0][:k], j_b=arrs[1][:k], n_a=arrs[2][:k], n_b=arrs[3][:k])

    def totals(self):
        arrs = [np.zeros(self.S, dtype=np.int64) for _ in range(4)]
        _chk(lib().lanesref_totals(self._h, *[_p(a, C.c_int64) for a in arrs]), "lanesref_totals")
        return dict(j_a=arrs[0], j_b=arrs[1], n_a=arrs[2], n_b=arrs[3])

    def profile(self):
        oa = np.zeros((self.S, self.L), dtype=np.uint32)
        ob = np.zeros((self.S, self.L), dtype=np.uint32)
        ns = C.c_int64()
        _chk(lib().lanesref_profile(self._h, _p(oa, C.c_uint32), _p(ob, C.c_uint32), C.byref(ns)),
             "lanesref_profile")
        return oa, ob, int(ns.value)


def unpack_words(words, L):
    """[S][nw] uint32 natural-layout words -> [S][L] uint8 sites (marshalling helper, no method arithmetic)."""
    w = np.ascontiguousarray(words, dtype=np.uint32)
    bits = np.unpackbits(w.view(np.uint8).reshape(w.shape[0], -1), axis=1, bitorder="little")
    return bits[:, :L]


def pack_sites(sites):
    """[S][L] uint8 sites -> [S][ceil(L/32)] uint32 natural-layout words."""
    s = np.ascontiguousarray(sites, dtype=np.uint8)
    S, L = s.shape
    pad = (-L) % 32
    if pad:
        s = np.concatenate([s, np.zeros((S, pad), dtype=np.uint8)], axis=1)
    return np.packbits(s, axis=1, bitorder="little").view(np.uint32).reshape(S, -1)


class Kpz2dRef:
    """The 2+1D generalisation (oracle/kpz2d_oracle.c)."""

    def __init__(self, Lx, Ly, nsamples, p, q, seed=0, first_sample=0, offset_mode=0):
        self.Lx, self.Ly, self.S = int(Lx), int(Ly), int(nsamples)
        self.row_words = (self.Lx + 31) // 32
        self._o = Options(int(first_sample), int(offset_mode), 0)
        self._h = C.c_void_p()
        self._nt = 0
        _chk(lib().kpz2dref_create(C.byref(self._h), C.c_int32(self.Lx), C.c_int32(self.Ly), C.c_int32(self.S),
                                   C.c_double(p), C.c_double(q), C.c_uint64(seed), C.byref(self._o)), "kpz2dref_create")

    def close(self):
        if getattr(self, "_h", None):
            lib().kpz2dref_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_record_times(self, t):
        t = _times(t)
        self._nt = len(t)
        _chk(lib().kpz2dref_set_record_times(self._h, _p(t, C.c_int64), C.c_int32(len(t))), "kpz2dref_set_record_times")

    def run(self, n_mcs):
        _chk(lib().kpz2dref_run(self._h, C.c_int64(n_mcs)), "kpz2dref_run")

    @property
    def time(self):
        t = C.c_int64()
        _chk(lib().kpz2dref_time(self._h, C.byref(t)), "kpz2dref_time")
        return t.value

    def slopes(self):
        sx = np.zeros((self.S, self.Ly, self.row_words), dtype=np.uint32)
        sy = np.zeros_like(sx)
        _chk(lib().kpz2dref_slopes(self._h, _p(sx, C.c_uint32), _p(sy, C.c_uint32)), "kpz2dref_slopes")
        return sx, sy

    def set_slopes(self, sx, sy):
        sx = np.ascontiguousarray(sx, dtype=np.uint32)
        sy = np.ascontiguousarray(sy, dtype=np.uint32)
        _chk(lib().kpz2dref_set_slopes(self._h, _p(sx, C.c_uint32), _p(sy, C.c_uint32)), "kpz2dref_set_slopes")

    def heights(self, sample):
        h = np.zeros((self.Ly, self.Lx), dtype=np.int32)
        _chk(lib().kpz2dref_heights(self._h, C.c_int32(sample), _p(h, C.c_int32)), "kpz2dref_heights")
        return h

    def roughness(self):
        cap = max(self._nt, 1)
        nt = C.c_int32(cap)
        t = np.zeros(cap, dtype=np.int64)
        s1 = np.zeros((cap, self.S), dtype=np.int64)
        s2 = np.zeros((cap, self.S), dtype=np.int64)
        w2 = np.zeros(cap, dtype=np.float64)
        _chk(lib().kpz2dref_roughness(self._h, C.byref(nt), _p(t, C.c_int64), _p(s1, C.c_int64), _p(s2, C.c_int64),
                                      _p(w2, C.c_double)), "kpz2dref_roughness")
        k = nt.value
        return dict(t=t[:k], sum_h=s1[:k], sum_h2=s2[:k], w2_mean=w2[:k])

    def hops(self):
        f = np.zeros(self.S, dtype=np.int64)
        b = np.zeros(self.S, dtype=np.int64)
        _chk(lib().kpz2dref_hops(self._h, _p(f, C.c_int64), _p(b, C.c_int64)), "kpz2dref_hops")
        return f, b
