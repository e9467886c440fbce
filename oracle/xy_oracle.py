"""ctypes view of oracle/xy_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It holds no arithmetic of the method: it compiles the C++ oracle with
g++ and marshals arguments.  It imports nothing from paper_1211_0780_b200.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "xy_oracle.cpp")
_LIB = os.path.join(_HERE, "libxy_oracle.so")
_lib = None


def build(force=False):
    """g++ -O2, no fast-math, no FMA contraction: libm double semantics are part of the definition."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", "-pthread", _SRC, "-o", _LIB]
    subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        vp, i32, u64 = C.c_void_p, C.c_int, C.c_uint64
        pd, pf, pi, pu32, pu64 = (C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int),
                                  C.POINTER(C.c_uint32), C.POINTER(C.c_uint64))
        sig = {
            "xyo_philox4x32_10": (None, [pu32, pu32, pu32]),
            "xyo_create": (vp, [i32, i32, pd, u64]),
            "xyo_destroy": (None, [vp]),
            "xyo_set_threads": (i32, [vp, i32]),
            "xyo_set_active_slots": (i32, [vp, pi, i32]),
            "xyo_init_random": (i32, [vp]),
            "xyo_init_ordered": (i32, [vp, C.c_float]),
            "xyo_state_ptr": (pf, [vp]),
            "xyo_set_state": (i32, [vp, pf]),
            "xyo_get_state": (i32, [vp, pf]),
            "xyo_get_perm": (i32, [vp, pi]),
            "xyo_set_perm": (i32, [vp, pi]),
            "xyo_get_beta_of_slot": (i32, [vp, pd]),
            "xyo_get_counters": (i32, [vp, pu32]),
            "xyo_set_counters": (i32, [vp, pu32]),
            "xyo_get_accept_counts": (i32, [vp, pu64, pu64]),
            "xyo_set_trace": (i32, [vp, pd, pf, pd, pd, pd]),
            "xyo_metropolis_pass": (i32, [vp, i32]),
            "xyo_metropolis_sweep": (i32, [vp]),
            "xyo_overrelax_pass": (i32, [vp, i32]),
            "xyo_overrelax_sweep": (i32, [vp]),
            "xyo_measure_slots": (i32, [vp, pd]),
            "xyo_measure": (i32, [vp, pd]),
            "xyo_measure_stiffness": (i32, [vp, pd]),
            "xyo_pt_exchange_with_E": (i32, [vp, pd]),
            "xyo_pt_exchange": (i32, [vp]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    o = np.zeros(4, dtype=np.uint32)
    lib().xyo_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(o, C.c_uint32))
    return o


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle call {what} failed with {rc}")


class XYOracle:
    """One (L, R) system on the CPU.  Method names mirror the C ABI of include/xy.h."""

    def __init__(self, L, R, betas, seed, threads=1):
        b = np.ascontiguousarray(betas, dtype=np.float64)
        assert b.shape == (R,)
        self.L, self.R, self.N = int(L), int(R), int(L) ** 3
        self._h = lib().xyo_create(self.L, self.R, _p(b, C.c_double), C.c_uint64(int(seed)))
        if not self._h:
            raise ValueError("xyo_create rejected its arguments")
        self._trace = {}
        self.set_threads(threads)

    def __del__(self):
        if getattr(self, "_h", None) and lib is not None:                # None during interpreter shutdown
            lib().xyo_destroy(self._h)
            self._h = None

    def set_threads(self, n):
        _chk(lib().xyo_set_threads(self._h, int(n)), "set_threads")

    def set_active_slots(self, slots=None):
        if slots is None or len(slots) == 0:
            _chk(lib().xyo_set_active_slots(self._h, None, 0), "set_active_slots")
        else:
            s = np.ascontiguousarray(slots, dtype=np.int32)
            _chk(lib().xyo_set_active_slots(self._h, _p(s, C.c_int), len(s)), "set_active_slots")

    def init_random(self):
        _chk(lib().xyo_init_random(self._h), "init_random")

    def init_ordered(self, theta0=0.0):
        _chk(lib().xyo_init_ordered(self._h, C.c_float(theta0)), "init_ordered")

    def state_view(self):
        """Zero-copy numpy view [R, L, L, L] (z, y, x) of the oracle's fp32 angles."""
        ptr = lib().xyo_state_ptr(self._h)
        return np.ctypeslib.as_array(ptr, shape=(self.R, self.L, self.L, self.L))

    def set_state(self, s):
        s = np.ascontiguousarray(s, dtype=np.float32)
        assert s.size == self.R * self.N
        _chk(lib().xyo_set_state(self._h, _p(s, C.c_float)), "set_state")

    def get_state(self):
        s = np.empty((self.R, self.L, self.L, self.L), dtype=np.float32)
        _chk(lib().xyo_get_state(self._h, _p(s, C.c_float)), "get_state")
        return s

    def get_perm(self):
        p = np.empty(self.R, dtype=np.int32)
        _chk(lib().xyo_get_perm(self._h, _p(p, C.c_int)), "get_perm")
        return p

    def set_perm(self, perm):
        p = np.ascontiguousarray(perm, dtype=np.int32)
        _chk(lib().xyo_set_perm(self._h, _p(p, C.c_int)), "set_perm")

    def get_beta_of_slot(self):
        b = np.empty(self.R, dtype=np.float64)
        _chk(lib().xyo_get_beta_of_slot(self._h, _p(b, C.c_double)), "get_beta_of_slot")
        return b

    def get_counters(self):
        n = np.empty(3, dtype=np.uint32)
        _chk(lib().xyo_get_counters(self._h, _p(n, C.c_uint32)), "get_counters")
        return n

    def set_counters(self, n):
        n = np.ascontiguousarray(n, dtype=np.uint32)
        assert n.shape == (3,)
        _chk(lib().xyo_set_counters(self._h, _p(n, C.c_uint32)), "set_counters")

    def get_accept_counts(self):
        met = np.zeros(self.R, dtype=np.uint64)
        pt = np.zeros(max(self.R - 1, 1), dtype=np.uint64)
        _chk(lib().xyo_get_accept_counts(self._h, _p(met, C.c_uint64), _p(pt, C.c_uint64)), "get_accept_counts")
        return met, pt[: self.R - 1]

    def enable_trace(self, met=False, overrelax=False, pt=False):
        """Allocate trace buffers the next passes fill: met_p/met_u [R,N], or_h [R,N], pt_p/pt_u [R-1]."""
        t = {}
        if met:
            t["met_p"] = np.full((self.R, self.L, self.L, self.L), np.nan, dtype=np.float64)
            t["met_u"] = np.full((self.R, self.L, self.L, self.L), np.nan, dtype=np.float32)
        if overrelax:
            t["or_h"] = np.full((self.R, self.L, self.L, self.L), np.nan, dtype=np.float64)
        if pt:
            t["pt_p"] = np.full(max(self.R - 1, 1), np.nan, dtype=np.float64)
            t["pt_u"] = np.full(max(self.R - 1, 1), np.nan, dtype=np.float64)
        self._trace = t
        g = lambda k, ct: _p(t[k], ct) if k in t else None
        _chk(lib().xyo_set_trace(self._h, g("met_p", C.c_double), g("met_u", C.c_float), g("or_h", C.c_double),
                                 g("pt_p", C.c_double), g("pt_u", C.c_double)), "set_trace")
        return t

    def metropolis_pass(self, colour):
        _chk(lib().xyo_metropolis_pass(self._h, int(colour)), "metropolis_pass")

    def metropolis_sweep(self):
        _chk(lib().xyo_metropolis_sweep(self._h), "metropolis_sweep")

    def overrelax_pass(self, colour):
        _chk(lib().xyo_overrelax_pass(self._h, int(colour)), "overrelax_pass")

    def overrelax_sweep(self):
        _chk(lib().xyo_overrelax_sweep(self._h), "overrelax_sweep")

    def measure(self):
        out = np.empty((self.R, 5), dtype=np.float64)
        _chk(lib().xyo_measure(self._h, _p(out, C.c_double)), "measure")
        return out

    def measure_stiffness(self):
        """[R, 6] = Cx, Cy, Cz, Sx, Sy, Sz by rank: the sums of cos / sin of the bond angle per direction (Eq. 6)."""
        out = np.empty((self.R, 6), dtype=np.float64)
        _chk(lib().xyo_measure_stiffness(self._h, _p(out, C.c_double)), "measure_stiffness")
        return out

    def measure_slots(self):
        out = np.full((self.R, 5), np.nan, dtype=np.float64)
        _chk(lib().xyo_measure_slots(self._h, _p(out, C.c_double)), "measure_slots")
        return out

    def pt_exchange(self, E_by_slot=None):
        if E_by_slot is None:
            _chk(lib().xyo_pt_exchange(self._h), "pt_exchange")
        else:
            e = np.ascontiguousarray(E_by_slot, dtype=np.float64)
            assert e.shape == (self.R,)
            _chk(lib().xyo_pt_exchange_with_E(self._h, _p(e, C.c_double)), "pt_exchange_with_E")

    def mcs(self):
        """one Metropolis sweep, one over-relaxation sweep, then one PT exchange.  The observables are
        reduced ONCE per step: the by-slot energies that xyo_measure_slots returns are handed to
        xyo_pt_exchange_with_E (xyo_pt_exchange would reduce every slot a second time).  Returns them by rank,
        as they were before the exchange (R14)."""
        self.metropolis_sweep()
        self.overrelax_sweep()
        by_slot = self.measure_slots()
        obs = by_slot[self.get_perm()]
        self.pt_exchange(by_slot[:, 0])
        return obs
