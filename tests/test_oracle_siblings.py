"""Pins for the oracle's same-level ghost exchange (a refinement boundary
uses the same ghost zones as an inter-process boundary). CPU only.

What fixes the expected values, none of it the exchange code itself:
  * decomposition invariance — a level cut into abutting boxes must reproduce the UNCUT level bit for bit (the
    uncut scheme is pinned by test_oracle_scheme.py): a cell's update reads the same numbers in the same order
    whether its neighbour lives in the same box or arrives through the exchange;
  * the exact quadratic solution u = r^2 + 3 t^2 (closed form) through a hierarchy whose level-1 boxes abut,
    touch only at an edge, or sit two cells apart (partial ghost overlap);
  * geometry: after a step every ghost cell that lies in a sibling's interior holds that sibling's value.
"""
import numpy as np
import pytest

from paper_2503_09629_b200 import workloads as wl

N0 = 24                      # level 0: 24^3, level 1 covers parent cells 6..18, level 2 sits in the x-high half
L1_LO, L1_N = 12, 24
L2 = wl.Box(2, (56, 52, 48), (8, 12, 16))  # nests (4 cells of margin) in a piece of every cut used below


def _pieces(cuts_x, cuts_y, cuts_z):
    """Level-1 boxes: the 24^3 region [12, 36)^3 cut at the given level-global indices."""
    def segs(cuts):
        e = [L1_LO] + list(cuts) + [L1_LO + L1_N]
        return list(zip(e[:-1], e[1:]))
    out = []
    for z0, z1 in segs(cuts_z):
        for y0, y1 in segs(cuts_y):
            for x0, x1 in segs(cuts_x):
                out.append(wl.Box(1, (x0, y0, z0), (x1 - x0, y1 - y0, z1 - z0)))
    return out


def _data(w, level, box, comp):
    """Smooth pulse + a deterministic ripple that depends on the LEVEL-GLOBAL index only, so that every
    decomposition of a level gets the same numbers."""
    x, y, z = w.centres(level, w.level_boxes(level).index(box))
    i = np.arange(box.lo[0], box.lo[0] + box.n[0])
    j = np.arange(box.lo[1], box.lo[1] + box.n[1])
    k = np.arange(box.lo[2], box.lo[2] + box.n[2])
    r2 = z[:, None, None] ** 2 + y[None, :, None] ** 2 + (x[None, None, :] - 0.1) ** 2
    rip = np.sin(12.9898 * i[None, None, :] + 78.233 * j[None, :, None] + 37.719 * k[:, None, None] + comp + level)
    return (1.0 if comp == 0 else 0.3) * np.exp(-r2 / 0.1) + 1e-3 * rip


def _run(oracle_mod, l1_boxes, sub, sigma, steps=2):
    boxes = [wl.Box(0, (0, 0, 0), (N0, N0, N0))] + list(l1_boxes) + [L2]
    w = wl.Workload("siblings", boxes, (N0, N0, N0), ko_sigma=sigma)
    H = oracle_mod.OracleHierarchy(w.boxes, w.domain_cells, 1, w.ghost, w.xlo, w.xhi, None, ko_sigma=sigma)
    for b in boxes:
        ib = w.level_boxes(b.level).index(b)
        for c in (0, 1):
            H.set_state(b.level, ib, c, _data(w, b.level, b, c))
    for _ in range(steps):
        H.step(w.dt_coarse, sub)
    return w, H


def _assemble_level1(w, H, comp):
    out = np.full((L1_N, L1_N, L1_N), np.nan)
    for ib, b in enumerate(w.level_boxes(1)):
        o = [b.lo[a] - L1_LO for a in range(3)]
        out[o[2]:o[2] + b.n[2], o[1]:o[1] + b.n[1], o[0]:o[0] + b.n[0]] = H.read(1, ib, comp)
    return out


@pytest.mark.parametrize("sigma", [0.0, 0.2])
@pytest.mark.parametrize("sub", [True, False])
def test_cut_level_reproduces_the_uncut_level_bit_for_bit(oracle_mod, sub, sigma):
    w0, H0 = _run(oracle_mod, _pieces([], [], []), sub, sigma)
    ref1 = [_assemble_level1(w0, H0, c) for c in (0, 1)]
    cuts = {"x halves": ([24], [], []), "z 8+16": ([], [], [20]), "x, y quarters": ([24], [22], []),
            "eight boxes": ([24], [20], [20])}
    for name, (cx, cy, cz) in cuts.items():
        w, H = _run(oracle_mod, _pieces(cx, cy, cz), sub, sigma)
        for c in (0, 1):
            assert np.array_equal(_assemble_level1(w, H, c), ref1[c]), (name, "level 1", c)
            assert np.array_equal(H.read(0, 0, c), H0.read(0, 0, c)), (name, "level 0", c)
            assert np.array_equal(H.read(2, 0, c), H0.read(2, 0, c)), (name, "level 2", c)


def test_the_exchange_matters(oracle_mod):
    """The pin above must be able to fail: without the exchange the seam ghosts are interpolated from the parent
    and the cut level differs from the uncut one at truncation level. Emulated with boxes the exchange does not
    connect: the two halves placed in DIFFERENT hierarchies see only prolonged ghosts."""
    w0, H0 = _run(oracle_mod, _pieces([], [], []), True, 0.0, steps=1)
    half = [wl.Box(1, (L1_LO, L1_LO, L1_LO), (12, L1_N, L1_N))]
    boxes = [wl.Box(0, (0, 0, 0), (N0, N0, N0))] + half
    w = wl.Workload("half", boxes, (N0, N0, N0))
    H = oracle_mod.OracleHierarchy(w.boxes, w.domain_cells, 1, w.ghost, w.xlo, w.xhi, None)
    for b in boxes:
        for c in (0, 1):
            H.set_state(b.level, 0, c, _data(w, b.level, b, c))
    H.step(w.dt_coarse, True)
    d = np.abs(H.read(1, 0, 0) - _assemble_level1(w0, H0, 0)[:, :, :12])
    assert d[:, :, :6].max() < 1e-12 and d[:, :, -1].max() > 1e-7   # far side identical, seam side not


@pytest.mark.parametrize("sigma", [0.0, 0.2])
@pytest.mark.parametrize("sub", [True, False])
def test_exact_quadratic_solution_through_touching_and_near_siblings(oracle_mod, sub, sigma):
    """u = x^2+y^2+z^2+3t^2, rho = 6t is reproduced to rounding by every operator of the scheme (see
    test_composite_scheme_exact_for_quadratic_solution) — copies included. Level 1: two boxes abutting on a
    face, one touching them only along an edge, one two cells away (only part of its ghost shell overlaps)."""
    n, o = 64, 16  # level 1 starts 20 parent cells from the periodic seam of level 0 (it travels 12 cells per step)
    l1 = [wl.Box(1, (24 + o, 24 + o, 24 + o), (16, 24, 24)), wl.Box(1, (40 + o, 24 + o, 24 + o), (16, 24, 24)),
          wl.Box(1, (56 + o, 48 + o, 24 + o), (12, 16, 24)), wl.Box(1, (24 + o, 50 + o, 24 + o), (30, 14, 24))]
    boxes = [wl.Box(0, (0, 0, 0), (n, n, n))] + l1 + [wl.Box(2, (88 + 2 * o, 60 + 2 * o, 60 + 2 * o), (16, 16, 16))]
    w = wl.Workload("quadratic siblings", boxes, (n, n, n), init=wl.quadratic_init, ko_sigma=sigma)
    H = oracle_mod.OracleHierarchy.from_workload(w)
    H.step(w.dt_coarse, sub)
    t = w.dt_coarse
    for l in (1, 2):
        for ib in range(len(w.level_boxes(l))):
            for c in (0, 1):
                got = H.read(l, ib, c, padded=True)
                want = wl.quadratic_exact(w, l, ib, c, t, pad=w.ghost)
                assert np.max(np.abs(got - want)) < 3e-12, (sub, l, ib, c, float(np.max(np.abs(got - want))))


def test_ghosts_inside_a_sibling_hold_the_siblings_values(oracle_mod):
    w, H = _run(oracle_mod, _pieces([24], [22], []), True, 0.0, steps=1)
    g = w.ghost
    lb = w.level_boxes(1)
    checked = 0
    for ia, A in enumerate(lb):
        pa = H.read(1, ia, 0, padded=True)
        for ib, B in enumerate(lb):
            if ia == ib:
                continue
            lo = [max(A.lo[a] - g, B.lo[a]) for a in range(3)]
            hi = [min(A.lo[a] + A.n[a] + g, B.lo[a] + B.n[a]) for a in range(3)]
            if any(h <= l for l, h in zip(lo, hi)):
                continue
            yb = H.read(1, ib, 0)
            sa = tuple(slice(lo[a] - A.lo[a] + g, hi[a] - A.lo[a] + g) for a in (2, 1, 0))
            sb = tuple(slice(lo[a] - B.lo[a], hi[a] - B.lo[a]) for a in (2, 1, 0))
            assert np.array_equal(pa[sa], yb[sb]), (ia, ib)
            checked += 1
    assert checked == 12  # 4 boxes x (2 face + 1 edge neighbours)


def test_overlapping_siblings_are_rejected(oracle_mod):
    boxes = [wl.Box(0, (0, 0, 0), (N0, N0, N0)), wl.Box(1, (12, 12, 12), (14, 24, 24)),
             wl.Box(1, (24, 12, 12), (12, 24, 24))]
    with pytest.raises(ValueError, match="overlap"):
        oracle_mod.OracleHierarchy(boxes, (N0, N0, N0))
