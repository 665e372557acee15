"""Element-by-element comparison of a hierarchy with the oracle — TEST INFRASTRUCTURE (see oracle.cpp).

One helper for `tests/test_gpu_*.py` and `__graft_entry__.smoke()`, so that the tolerance is written once.
The object under test is passed in (anything with `sc_debug_read_padded` / `sc_read_level`); nothing here
imports the CUDA package.

Tolerance (BASELINE.json north_star): max|delta| <= 1e-11 * max|u| in fp64, read PER COMPONENT TYPE (DESIGN.md
section 4, reading S27):
  u components:   |delta| <= 1e-11 * max|u|     (max over the u components of all levels, boxes and fields, oracle
                                                 values, interiors) — exactly as stated; u is never given rho's scale;
  rho components: |delta| <= 1e-11 * max|rho| + F,   F = nsteps * 4 * 2^(L-1) * 2^-53 * (0.625 / dx_finest) * max|u|.
  over n > 1 coarse steps the floor of rho accumulates (n F) and feeds u through u += dt rho:  the u bound gains
  F_u(n) = dt_coarse * F(1) * n (n + 1) / 2  (7e-14 max|u| for n = 1 at cfg 5's depth: nothing; 1.4e-11 for its 20 steps), with
  max|u| in F taken over the run (`floor_scale`: the pulse of cfg 5 decays to 0.3 of its initial height).
F is the rounding floor of the DEFINITION, not an allowance for the kernels: one RHS evaluation forms Lap_h u from
terms of size 30 |u| / (12 dx^2), so rho = d_t u is rounded by eps * 2.5 |u| dt / dx^2 = eps * 0.625 |u| / dx per
evaluation (dt = dx / 4), and the finest of L levels is evaluated 4 * 2^(L-1) times per coarse step. For shallow
hierarchies F is nothing (3 levels of 32^3: 7e-14); at cfg 5's depth (dx = 2 / 8192, 128 evaluations) it is 3.5e-11 max|u|,
above 1e-11 * max|rho| after one step from rho = 0. That the floor is real and not a kernel defect is MEASURED at that
depth without any kernel (tests/test_oracle_scheme.py::test_rounding_floor_of_the_oracle, S27): on six levels with
cfg 5's dx and dt the fp64 oracle lies 7.0e-12 max|u| in rho (7e-16 in u) from the oracle built in long double, and its
plain and FMA-contracted fp64 builds lie 9.3e-12 max|u| apart. F covers the measured distance five times. How close the
CUDA path is to that long double value is tests/test_gpu_truth.py (2.0-2.4e-11 at cfg 5's depth; GPU - oracle = 0.67 F).
"""
from __future__ import annotations

import numpy as np

RTOL = 1e-11


def u_scale(O, w) -> float:
    """max|u| over the u components (comp < nfields) of every box of every level, from the oracle."""
    s = 0.0
    for l in range(w.nlevels):
        for ib in range(len(w.level_boxes(l))):
            for c in range(w.nfields):
                s = max(s, float(np.max(np.abs(O.read_level(l, ib, c)))))
    return s


def rho_scale(O, w) -> float:
    """max|rho| over the rho components (comp >= nfields), from the oracle. May be 0 (rho = 0 initial data, no step
    taken): compare_state uses max(rho_scale, u_scale)."""
    s = 0.0
    for l in range(w.nlevels):
        for ib in range(len(w.level_boxes(l))):
            for c in range(w.nfields, w.ncomp):
                s = max(s, float(np.max(np.abs(O.read_level(l, ib, c)))))
    return s


def rho_floor(w, su: float, nsteps: int = 1) -> float:
    """F of the module docstring: accumulated rounding of rho on the finest level over `nsteps` coarse steps."""
    L = w.nlevels
    return nsteps * 4.0 * (1 << (L - 1)) * 2.0 ** -53 * (0.625 / w.dx(L - 1)) * su


def u_floor(w, su: float, nsteps: int = 1) -> float:
    """F_u of the module docstring: what the accumulated rounding of rho adds to u over `nsteps` coarse steps."""
    return w.dt_coarse * rho_floor(w, su, 1) * nsteps * (nsteps + 1) / 2.0


def compare_state(G, O, w, padded: bool = True, what: str = "state", rtol: float = RTOL, levels=None,
                  nsteps: int = 1, floor_scale: float = 0.0) -> float:
    """Assert the tolerance of the module docstring for every component of every box (ghosts included if `padded`);
    returns the worst difference in units of its component type's bound / rtol. One array pair is alive at a time.
    `nsteps`: coarse steps taken since the two states were equal (only scales the rounding floors; the default 1 is
    the strictest); `floor_scale`: max|u| over the run if it was larger than it is now."""
    su = u_scale(O, w)
    assert su > 0.0 and np.isfinite(su), (what, su)
    fs = max(su, floor_scale)
    tol_u = rtol * su + u_floor(w, fs, nsteps)
    tol_r = rtol * max(rho_scale(O, w), su) + rho_floor(w, fs, nsteps)
    worst = 0.0
    for l in (range(w.nlevels) if levels is None else levels):
        for ib in range(len(w.level_boxes(l))):
            for c in range(w.ncomp):
                a = G.sc_debug_read_padded(l, ib, c) if padded else G.sc_read_level(l, ib, c)
                assert np.isfinite(a).all(), (what, l, ib, c)
                b = O.read(l, ib, c, padded=padded)
                d = float(np.max(np.abs(a - b)))
                del a, b
                tol = tol_u if c < w.nfields else tol_r
                worst = max(worst, d / tol * rtol)
                assert d <= tol, \
                    f"{what}: level {l} box {ib} comp {c}: max|d| = {d:.3e} > {tol:.3e} ({'u' if c < w.nfields else 'rho'} bound)"
    return worst
