"""ctypes wrapper around oracle/flatspin_oracle.cpp -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this package.  The product (paper_2002_11401_b200) never does.  See the header of
flatspin_oracle.cpp for what the oracle computes and what pins it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "flatspin_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (fp64, no FMA contraction so it rounds like the formulas read)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c++17", "-shared", "-fPIC",
                               _SRC, "-o", _LIB])
    return _LIB


class _Params(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("alpha", "b", "c", "beta", "gamma", "neighbor_distance")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int, C.c_double
        P = C.POINTER
        L.orc_create.restype = vp
        L.orc_create.argtypes = [i64, vp, vp, vp, P(_Params), i32]
        L.orc_destroy.argtypes = [vp]
        for name in ("orc_build_neighbors", "orc_guard_violations", "orc_coincident", "orc_num_interactions"):
            getattr(L, name).restype = i64
            getattr(L, name).argtypes = [vp]
        L.orc_get_neighbors.argtypes = [vp, vp, i64]
        L.orc_neighbors_of.restype = i64
        L.orc_neighbors_of.argtypes = [vp, i64, vp, i64]
        L.orc_set_spins.argtypes = [vp, vp]
        L.orc_get_spins.argtypes = [vp, vp]
        L.orc_set_thermal.argtypes = [vp, dbl, C.c_uint64]
        L.orc_set_field.argtypes = [vp, dbl, dbl, C.c_uint32]
        L.orc_set_local_field.argtypes = [vp, vp]
        L.orc_coupling.argtypes = [vp, i64, i64, vp]
        L.orc_field_one.argtypes = [vp, i64, i32, vp]
        L.orc_fields.argtypes = [vp, i32, vp]
        L.orc_key_one.restype = dbl
        L.orc_key_one.argtypes = [vp, i64]
        L.orc_scan.argtypes = [vp, P(i64), P(i64), P(dbl)]
        for name in ("orc_relax_A", "orc_relax_B"):
            getattr(L, name).restype = i64
            getattr(L, name).argtypes = [vp, i64, vp, i64]
        L.orc_cached_hdip.argtypes = [vp, vp]
        L.orc_gather_cached.argtypes = [vp]
        L.orc_set_threads.argtypes = [vp, i32]
        L.orc_build_weights.argtypes = [vp]
        L.orc_scan_cached.argtypes = [vp, P(i64), P(i64), P(dbl)]
        L.orc_monitor.argtypes = [vp, P(i64), P(dbl), P(dbl), i32]
        L.orc_spin_correlation.argtypes = [vp, dbl, i64, vp, vp]
        L.orc_vertex_populations.argtypes = [vp, vp, i64, vp]
        L.orc_energy.restype = dbl
        L.orc_energy.argtypes = [vp]
        L.orc_astroid_L.restype = dbl
        L.orc_astroid_L.argtypes = [dbl, dbl, dbl, P(_Params)]
        L.orc_philox.argtypes = [vp, vp, vp]
        L.orc_unit_normals.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, vp]
        _lib = L
    return _lib


def _params(d) -> _Params:
    return _Params(d["alpha"], d["b"], d["c"], d["beta"], d["gamma"], d["neighbor_distance"])


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32); k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, np.uint32)
    lib().orc_philox(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out


def unit_normals(seed, step, spin):
    z = np.zeros(2)
    lib().orc_unit_normals(int(seed), int(step), int(spin), z.ctypes.data)
    return z


def astroid_L(hpar, hperp, hk, params):
    p = _params(params)
    return lib().orc_astroid_L(float(hpar), float(hperp), float(hk), C.byref(p))


class Oracle:
    """One ASI system held by the CPU oracle."""

    def __init__(self, pos, angle, hc, params, spins=None, brute_force_neighbors=False):
        self.L = lib()
        pos = np.ascontiguousarray(pos, np.float64); angle = np.ascontiguousarray(angle, np.float64)
        hc = np.ascontiguousarray(hc, np.float64)
        self.N = int(angle.shape[0])
        assert pos.shape == (self.N, 2) and hc.shape == (self.N,)
        self._p = _params(params)
        self.h = self.L.orc_create(self.N, pos.ctypes.data, angle.ctypes.data, hc.ctypes.data,
                                   C.byref(self._p), int(brute_force_neighbors))
        if spins is not None:
            self.set_spins(spins)

    def __del__(self):
        if getattr(self, "h", None):
            self.L.orc_destroy(self.h); self.h = None

    def build_neighbors(self) -> int:
        return int(self.L.orc_build_neighbors(self.h))

    @property
    def guard_violations(self): return int(self.L.orc_guard_violations(self.h))
    @property
    def coincident(self): return int(self.L.orc_coincident(self.h))
    @property
    def num_interactions(self): return int(self.L.orc_num_interactions(self.h))

    def neighbors(self):
        K = self.build_neighbors()
        out = np.full((self.N, max(K, 1)), -1, np.int32)
        self.L.orc_get_neighbors(self.h, out.ctypes.data, max(K, 1))
        return out[:, :K] if K else out[:, :0]

    def neighbors_of(self, i, cap=1 << 16):
        out = np.zeros(cap, np.int32)
        n = int(self.L.orc_neighbors_of(self.h, int(i), out.ctypes.data, cap))
        return out[:n].copy()

    def set_spins(self, s):
        s = np.ascontiguousarray(s, np.int8); assert s.shape == (self.N,)
        self.L.orc_set_spins(self.h, s.ctypes.data)

    def spins(self):
        s = np.zeros(self.N, np.int8); self.L.orc_get_spins(self.h, s.ctypes.data); return s

    def set_thermal(self, sigma, seed): self.L.orc_set_thermal(self.h, float(sigma), int(seed))
    def set_field(self, hx, hy, step=0): self.L.orc_set_field(self.h, float(hx), float(hy), int(step))

    def set_local_field(self, h):
        """Per-spin external field [N,2] (global x,y components) added to the global one; None clears."""
        if h is None:
            self.L.orc_set_local_field(self.h, None); return
        h = np.ascontiguousarray(h, np.float64); assert h.shape == (self.N, 2)
        self.L.orc_set_local_field(self.h, h.ctypes.data)

    def coupling(self, i, j):
        g = np.zeros(2); self.L.orc_coupling(self.h, int(i), int(j), g.ctypes.data); return g

    def field_one(self, i, which=0):
        h = np.zeros(2); self.L.orc_field_one(self.h, int(i), int(which), h.ctypes.data); return h

    def fields(self, which=0):
        h = np.zeros((self.N, 2)); self.L.orc_fields(self.h, int(which), h.ctypes.data); return h

    def key_one(self, i): return float(self.L.orc_key_one(self.h, int(i)))

    def scan(self):
        n, b, l = C.c_int64(), C.c_int64(), C.c_double()
        self.L.orc_scan(self.h, C.byref(n), C.byref(b), C.byref(l))
        return n.value, b.value, l.value

    def _relax(self, fn, max_flips, cap):
        cap = int(cap if cap is not None else 4 * self.N + 1024)
        log = np.zeros(cap, np.int32)
        n = int(fn(self.h, int(max_flips), log.ctypes.data, cap))
        return n, log[:min(n, cap)].copy()

    def relax_A(self, max_flips=0, cap=None): return self._relax(self.L.orc_relax_A, max_flips, cap)
    def relax_B(self, max_flips=0, cap=None): return self._relax(self.L.orc_relax_B, max_flips, cap)

    def cached_hdip(self):
        h = np.zeros((self.N, 2)); self.L.orc_cached_hdip(self.h, h.ctypes.data); return h

    def gather_cached(self): self.L.orc_gather_cached(self.h)
    def build_weights(self): self.L.orc_build_weights(self.h)
    def set_threads(self, n): self.L.orc_set_threads(self.h, int(n))

    def scan_cached(self):
        n, b, l = C.c_int64(), C.c_int64(), C.c_double()
        self.L.orc_scan_cached(self.h, C.byref(n), C.byref(b), C.byref(l))
        return n.value, b.value, l.value

    def monitor(self, reset=False):
        n, g, t = C.c_int64(), C.c_double(), C.c_double()
        self.L.orc_monitor(self.h, C.byref(n), C.byref(g), C.byref(t), int(reset))
        return n.value, g.value, t.value

    def energy(self): return float(self.L.orc_energy(self.h))

    def spin_correlation(self, bin_width, nbins):
        """(sum of c_ij, number of pairs) per separation bin floor(|r_ij| / bin_width)."""
        sm = np.zeros(nbins, np.int64); cnt = np.zeros(nbins, np.int64)
        self.L.orc_spin_correlation(self.h, float(bin_width), int(nbins), sm.ctypes.data, cnt.ctypes.data)
        return sm, cnt

    def vertex_populations(self, vertices):
        """Counts of Type I, II, III, IV vertices; vertices [V,4] spin indices."""
        v = np.ascontiguousarray(vertices, np.int32); assert v.ndim == 2 and v.shape[1] == 4
        out = np.zeros(4, np.int64)
        self.L.orc_vertex_populations(self.h, v.ctypes.data, int(v.shape[0]), out.ctypes.data)
        return out
