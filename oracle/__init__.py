"""CPU oracle — TEST INFRASTRUCTURE ONLY (see the header of oracle.cpp).

ctypes wrapper around ``liboracle.so`` (built from ``oracle.cpp`` by :func:`build`). May be imported only
by ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs.
It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# ORACLE_SO / ORACLE_CXXFLAGS: build and load a VARIANT of the same source (tests only: the rounding-floor pin compares
# the default build with one that contracts multiply-adds, tests/test_oracle_scheme.py)
_SO = os.environ.get("ORACLE_SO") or os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "oracle.cpp")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle.cpp with g++ (-O2, OpenMP, no fast-math)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra"] + \
              os.environ.get("ORACLE_CXXFLAGS", "").split() + ["-o", _SO, _SRC]
        subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.oc_last_error.restype = C.c_char_p
        L.oc_set_threads.argtypes = [C.c_int]
        L.oc_max_threads.restype = C.c_int
        L.oc_b.restype = C.c_double
        L.oc_b.argtypes = [C.c_int, C.c_int, C.c_double]
        L.oc_dense_stage.restype = C.c_double
        L.oc_dense_stage.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, dp]
        L.oc_prolong_weights.argtypes = [C.c_int, dp]
        L.oc_restrict_weights.argtypes = [dp]
        L.oc_create.restype = C.c_void_p
        L.oc_create.argtypes = [C.c_int, C.c_int, ip, ip, ip, C.c_int, C.c_int, ip, dp, dp, dp]
        L.oc_destroy.argtypes = [C.c_void_p]
        L.oc_set_dissipation.argtypes = [C.c_void_p, C.c_double]
        L.oc_set_fd_order.argtypes = [C.c_void_p, C.c_int]
        L.oc_set_options.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
        L.oc_interp_weights.argtypes = [C.c_int, C.c_int, ip, ip, dp, dp, ip, ip, dp]
        L.oc_b_rk.restype = C.c_double
        L.oc_b_rk.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double]
        L.oc_dense_stage_rk.restype = C.c_double
        L.oc_dense_stage_rk.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, dp]
        L.oc_set_state.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, dp]
        L.oc_read.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, dp]
        L.oc_step.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.oc_time.restype = C.c_double
        L.oc_time.argtypes = [C.c_void_p]
        L.oc_ghost_map.restype = C.c_longlong
        L.oc_ghost_map.argtypes = [C.c_void_p, C.c_int, C.c_int, ip, C.c_ulonglong]
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def b(i: int, m: int, theta: float) -> float:
    return lib().oc_b(i, m, theta)


def dense_stage(stage: int, theta: float, hp: float, y_old: float, k: Sequence[float]) -> float:
    kk = np.ascontiguousarray(k, dtype=np.float64)
    return lib().oc_dense_stage(stage, theta, hp, y_old, _dp(kk))


def prolong_weights(parity: int) -> np.ndarray:
    w = np.zeros(5)
    lib().oc_prolong_weights(parity, _dp(w))
    return w


def restrict_weights() -> np.ndarray:
    r = np.zeros(6)
    lib().oc_restrict_weights(_dp(r))
    return r


def b_rk(integrator: int, i: int, m: int, theta: float) -> float:
    """m-th theta-derivative of the dense-output polynomial b_i of RK4 (4), Kutta's RK3 (3) or midpoint RK2 (2)."""
    return lib().oc_b_rk(integrator, i, m, theta)


def dense_stage_rk(integrator: int, stage: int, theta: float, hp: float, y_old: float, k: Sequence[float]) -> float:
    kk = np.zeros(4)
    kk[:len(k)] = k
    return lib().oc_dense_stage_rk(integrator, stage, theta, hp, y_old, _dp(kk))


def interp_weights(interp: int = 0, vertex: int = 0):
    """(omin, w[2][np], rmin, r[nr]) of the prolongation / restriction operators (oracle.cpp: make_interp)."""
    w0, w1, r = np.zeros(10), np.zeros(10), np.zeros(10)
    n = (C.c_int * 4)()
    I = C.POINTER(C.c_int)
    at = lambda q: C.cast(C.byref(n, 4 * q), I)  # noqa: E731
    lib().oc_interp_weights(interp, vertex, at(0), at(1), _dp(w0), _dp(w1), at(2), at(3), _dp(r))
    return n[1], np.stack([w0[:n[0]], w1[:n[0]]]), n[3], r[:n[2]].copy()


def set_threads(n: int) -> None:
    lib().oc_set_threads(n)


def max_threads() -> int:
    return lib().oc_max_threads()


class OracleHierarchy:
    """Same role as the CUDA binding's Hierarchy, on the CPU. ``boxes``: sequence of objects with
    ``level``, ``lo``, ``n`` (x, y, z)."""

    SLOT_Y, SLOT_YOLD, SLOT_K1 = 0, 1, 2

    def __init__(self, boxes, domain_cells, nfields: int = 1, ghost: int = 3,
                 xlo=(-1.0, -1.0, -1.0), xhi=(1.0, 1.0, 1.0), coupling: Optional[np.ndarray] = None,
                 ko_sigma: float = 0.0, fd_order: int = 4, integrator: int = 4, outer_bc: int = 0, ko_order: int = 0,
                 interp: int = 0, vertex: int = 0):
        L = lib()
        self.boxes = list(boxes)
        self.nfields, self.ghost = nfields, ghost
        lev = np.array([bx.level for bx in self.boxes], dtype=np.int32)
        lo = np.array([bx.lo for bx in self.boxes], dtype=np.int32).reshape(-1)
        n = np.array([bx.n for bx in self.boxes], dtype=np.int32).reshape(-1)
        dom = np.array(domain_cells, dtype=np.int32)
        xl, xh = np.array(xlo, dtype=np.float64), np.array(xhi, dtype=np.float64)
        cp = None
        if coupling is not None:
            cmat = np.ascontiguousarray(coupling, dtype=np.float64)
            assert cmat.shape == (nfields, nfields)
            cp = _dp(cmat)
        nlev = int(lev.max()) + 1 if len(lev) else 0
        self._h = L.oc_create(nlev, len(self.boxes), _ip(lev), _ip(lo), _ip(n), ghost, nfields, _ip(dom),
                              _dp(xl), _dp(xh), cp)
        if not self._h:
            raise ValueError("oracle: " + L.oc_last_error().decode())
        self.nlevels = nlev
        if fd_order != 4 and L.oc_set_fd_order(self._h, int(fd_order)) != 0:
            raise ValueError("oracle: " + L.oc_last_error().decode())
        # always: ko_order = 0 resolves to eq 36's r = fd_order, which depends on the call above
        if L.oc_set_options(self._h, int(integrator), int(outer_bc), int(ko_order), int(interp), int(vertex)) != 0:
            raise ValueError("oracle: " + L.oc_last_error().decode())
        if ko_sigma and L.oc_set_dissipation(self._h, float(ko_sigma)) != 0:
            raise ValueError("oracle: " + L.oc_last_error().decode())

    @classmethod
    def from_workload(cls, w) -> "OracleHierarchy":
        h = cls(w.boxes, w.domain_cells, w.nfields, w.ghost, w.xlo, w.xhi, w.coupling,
                ko_sigma=getattr(w, "ko_sigma", 0.0), fd_order=getattr(w, "fd_order", 4),
                integrator=getattr(w, "integrator", 4), outer_bc=getattr(w, "outer_bc", 0),
                ko_order=getattr(w, "ko_order", 0), interp=getattr(w, "interp", 0), vertex=int(getattr(w, "vertex", 0)))
        for l in range(w.nlevels):
            for ib in range(len(w.level_boxes(l))):
                for c in range(w.ncomp):
                    h.set_state(l, ib, c, w.initial_state(l, ib, c))
        return h

    def _box(self, level: int, ibox: int):
        return [bx for bx in self.boxes if bx.level == level][ibox]

    def set_state(self, level: int, ibox: int, comp: int, arr: np.ndarray) -> None:
        bx = self._box(level, ibox)
        a = np.ascontiguousarray(arr, dtype=np.float64)
        assert a.size == bx.n[0] * bx.n[1] * bx.n[2]
        if lib().oc_set_state(self._h, level, ibox, comp, _dp(a)) != 0:
            raise ValueError("oracle: set_state")

    def read(self, level: int, ibox: int, comp: int, slot: int = 0, padded: bool = False) -> np.ndarray:
        bx = self._box(level, ibox)
        e = self.ghost if padded else 0
        out = np.empty((bx.n[2] + 2 * e, bx.n[1] + 2 * e, bx.n[0] + 2 * e), dtype=np.float64)
        if lib().oc_read(self._h, level, ibox, slot, comp, int(padded), _dp(out)) != 0:
            raise ValueError("oracle: read")
        return out

    def read_level(self, level: int, ibox: int, comp: int) -> np.ndarray:
        return self.read(level, ibox, comp)

    def step(self, dt_coarse: float, subcycling: bool = True) -> None:
        if lib().oc_step(self._h, dt_coarse, int(subcycling)) != 0:
            raise ValueError("oracle: step")

    @property
    def time(self) -> float:
        return lib().oc_time(self._h)

    def ghost_map(self, level: int, ibox: int) -> np.ndarray:
        n = lib().oc_ghost_map(self._h, level, ibox, None, 0)
        if n < 0:
            raise ValueError("oracle: ghost_map")
        out = np.empty((n, 7), dtype=np.int32)
        lib().oc_ghost_map(self._h, level, ibox, _ip(out), out.size)
        return out

    def close(self) -> None:
        if getattr(self, "_h", None):
            lib().oc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


if __name__ == "__main__":
    print(build(force=True))
