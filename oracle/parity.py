"""Element-by-element comparison of a hierarchy with the oracle — TEST INFRASTRUCTURE (see oracle.cpp).

One helper for `tests/test_gpu_*.py` and `__graft_entry__.smoke()`, so that the tolerance is written once.
The object under test is passed in (anything with `sc_debug_read_padded` / `sc_read_level`); nothing here
imports the CUDA package.

Tolerance (BASELINE.json north_star): max|delta| <= 1e-11 * max|u| in fp64, where max|u| is taken over the u
components only (all levels, boxes and fields, oracle values, interiors) and the bound is applied to EVERY
component, ghosts included: rho = d_t u is usually the larger quantity (max|rho| ~ 20 max|u| for the narrow
pulses of cfg 3/5), so this is the strict reading — u is never given rho's scale.
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


def compare_state(G, O, w, padded: bool = True, what: str = "state", rtol: float = RTOL, levels=None) -> float:
    """Assert |G - O| <= rtol * max|u| for every component of every box (ghosts included if `padded`);
    returns the worst difference in units of max|u|. One array pair is alive at a time."""
    scale = u_scale(O, w)
    assert scale > 0.0 and np.isfinite(scale), (what, scale)
    worst = 0.0
    for l in (range(w.nlevels) if levels is None else levels):
        for ib in range(len(w.level_boxes(l))):
            for c in range(w.ncomp):
                a = G.sc_debug_read_padded(l, ib, c) if padded else G.sc_read_level(l, ib, c)
                assert np.isfinite(a).all(), (what, l, ib, c)
                b = O.read(l, ib, c, padded=padded)
                d = float(np.max(np.abs(a - b)))
                del a, b
                worst = max(worst, d)
                assert d <= rtol * scale, \
                    f"{what}: level {l} box {ib} comp {c}: max|d| = {d:.3e} > {rtol:g} * max|u| = {rtol * scale:.3e}"
    return worst / scale
