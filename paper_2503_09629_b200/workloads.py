"""Seeded synthetic workloads: the five BASELINE.json configurations as box lists plus initial data.

This module holds NONE of the method's arithmetic (no RK4, no dense output, no stencils, no
interpolation weights): it only describes hierarchies and produces input arrays. It is the one module
that both the CUDA path's tests/bench and the CPU oracle's tests import (numpy only; it imports
neither the CUDA binding nor anything under ``oracle/``).

Shapes follow the paper's own workloads (PAPER.md:236 three-level scalar-wave box-in-box grid;
PAPER.md:248-254 nine-level BBH box-in-box grid with 22 evolved fields) as bracketed by
BASELINE.json's ``configs``; the concrete numbers are SURVEY.md section 8(d) "Configs as concrete inputs"
and the readings S17-S23 restated in DESIGN.md.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Callable, List, Optional, Sequence, Tuple

import numpy as np

SEED = 250309629
GHOST = 3
CFL = 0.25

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


# ----------------------------------------------------------------------------------------------
# counter-based random numbers (splitmix64 finaliser), vectorised; no state, any order of evaluation
# ----------------------------------------------------------------------------------------------
def _mix64(z: np.ndarray) -> np.ndarray:
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        z = z ^ (z >> np.uint64(31))
    return z


def _key(seed: int, *ids: int) -> np.uint64:
    k = _mix64(np.uint64(seed & 0xFFFFFFFFFFFFFFFF))
    for i in ids:
        k = _mix64(k ^ np.uint64(int(i) & 0xFFFFFFFFFFFFFFFF))
    return np.uint64(k)


def counter_uniform01(seed: int, ids: Sequence[int], counters: np.ndarray) -> np.ndarray:
    """U[0,1) doubles (53-bit) as a pure function of (seed, ids, counter)."""
    k = _key(seed, *ids)
    z = _mix64(np.asarray(counters, dtype=np.uint64) ^ k)
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def counter_normal(seed: int, ids: Sequence[int], counters: np.ndarray) -> np.ndarray:
    """N(0,1) by Box-Muller on two counter streams (reading S21)."""
    c = np.asarray(counters, dtype=np.uint64)
    u1 = counter_uniform01(seed, list(ids) + [1], c)
    u2 = counter_uniform01(seed, list(ids) + [2], c)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * math.pi * u2)


# ----------------------------------------------------------------------------------------------
# hierarchy description
# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass(frozen=True)
class Box:
    level: int
    lo: Tuple[int, int, int]  # (x, y, z) first interior cell, level-global index
    n: Tuple[int, int, int]   # (x, y, z) interior cells


@dataclasses.dataclass
class Workload:
    name: str
    boxes: List[Box]
    domain_cells: Tuple[int, int, int]
    nfields: int = 1
    ghost: int = GHOST
    xlo: Tuple[float, float, float] = (-1.0, -1.0, -1.0)
    xhi: Tuple[float, float, float] = (1.0, 1.0, 1.0)
    coupling: Optional[np.ndarray] = None      # (F, F) or None
    coarse_steps: int = 1
    init: Optional[Callable[["Workload", int, int, int], np.ndarray]] = None
    note: str = ""
    ko_sigma: float = 0.0                      # Kreiss-Oliger strength (eqs 35-36); 0 = none
    fd_order: int = 4                          # centred finite differences of the RHS: 4 (S2) or 8 (ghost >= 4)
    integrator: int = 4                        # 4: RK4; 3: Kutta's RK3; 2: midpoint RK2 (reading S28)
    outer_bc: int = 0                          # level 0: 0 periodic (S9); 1 radiative / Sommerfeld
    ko_order: int = 0                          # 0: eq 36's r = fd_order; 5: delta^6 (3 ghost layers); 9: delta^10 (5)
    interp: int = 0                            # 0: quartic / quintic (S3, S4); 1: 9-point / 10-point (follows fd_order 8)
    vertex: int = 0                            # 1: vertex-centred grids, injection restriction (S31)

    @property
    def nlevels(self) -> int:
        return max(b.level for b in self.boxes) + 1

    @property
    def ncomp(self) -> int:
        return 2 * self.nfields

    def dx(self, level: int) -> float:
        return (self.xhi[0] - self.xlo[0]) / (self.domain_cells[0] * (1 << level))

    @property
    def dt_coarse(self) -> float:
        return CFL * self.dx(0)

    def level_boxes(self, level: int) -> List[Box]:
        return [b for b in self.boxes if b.level == level]

    def box(self, level: int, ibox: int) -> Box:
        return self.level_boxes(level)[ibox]

    def centres(self, level: int, ibox: int, pad: int = 0):
        """Cell-centre (grid-point, for vertex-centred grids) coordinate vectors (x, y, z) of a box, optionally
        padded by ``pad`` cells."""
        b = self.box(level, ibox)
        out = []
        for a in range(3):
            d = (self.xhi[a] - self.xlo[a]) / (self.domain_cells[a] * (1 << level))
            idx = np.arange(b.lo[a] - pad, b.lo[a] + b.n[a] + pad, dtype=np.float64)
            out.append(self.xlo[a] + (idx + (0.0 if self.vertex else 0.5)) * d)
        return out

    def initial_state(self, level: int, ibox: int, comp: int) -> np.ndarray:
        """Interior-only array [nz][ny][nx] (x fastest) for one component of one box."""
        assert self.init is not None
        return np.ascontiguousarray(self.init(self, level, ibox, comp), dtype=np.float64)

    # work accounting: one update = one interior cell of one box, all V arrays,
    # advanced by one RK4 level-step
    def cells(self, level: int) -> int:
        return sum(b.n[0] * b.n[1] * b.n[2] for b in self.level_boxes(level))

    def updates_per_coarse_step(self, subcycling: bool) -> int:
        L = self.nlevels
        if subcycling:
            return sum((1 << l) * self.cells(l) for l in range(L))
        return sum((1 << (L - 1)) * self.cells(l) for l in range(L))

    def zone_cycles_per_coarse_step(self) -> int:
        """Paper convention: as if every cell took the smallest step."""
        L = self.nlevels
        return sum((1 << (L - 1)) * self.cells(l) for l in range(L))


def nested_cubes(nlevels: int, n: int) -> List[Box]:
    """nlevels boxes of n^3 cells, each centred in the domain [0, n*2^l)^3 of its level."""
    out = []
    for l in range(nlevels):
        lo = (n * (1 << l) - n) // 2
        out.append(Box(l, (lo, lo, lo), (n, n, n)))
    return out


# ----------------------------------------------------------------------------------------------
# initial data
# ----------------------------------------------------------------------------------------------
def _noise(w: Workload, level: int, ibox: int, comp: int, amp: float) -> np.ndarray:
    """amp * U(-1,1) per interior cell, keyed on (seed, level, box, comp, i, j, k) (reading S18)."""
    b = w.box(level, ibox)
    nx, ny, nz = b.n
    cnt = np.arange(nx * ny * nz, dtype=np.uint64)
    u = counter_uniform01(SEED, [level, ibox, comp], cnt).reshape(nz, ny, nx)
    return amp * (2.0 * u - 1.0)


def _r2(w: Workload, level: int, ibox: int, centre=(0.0, 0.0, 0.0)) -> np.ndarray:
    x, y, z = w.centres(level, ibox)
    return ((z[:, None, None] - centre[2]) ** 2 + (y[None, :, None] - centre[1]) ** 2
            + (x[None, None, :] - centre[0]) ** 2)


def gaussian_init(denominator: float, noise: float = 1e-6):
    """u = exp(-r^2/denominator), rho = 0, plus seeded uniform noise on every component."""
    def f(w: Workload, level: int, ibox: int, comp: int) -> np.ndarray:
        b = w.box(level, ibox)
        if comp < w.nfields:
            v = np.exp(-_r2(w, level, ibox) / denominator)
        else:
            v = np.zeros((b.n[2], b.n[1], b.n[0]))
        if noise:
            v = v + _noise(w, level, ibox, comp, noise)
        return v
    return f


PLANE_L = 2.0
PLANE_K = 2.0 * math.pi / PLANE_L
PLANE_OMEGA = PLANE_K * math.sqrt(3.0)


def plane_wave_exact(w: Workload, level: int, ibox: int, comp: int, t: float) -> np.ndarray:
    """Exact solution u = sin(k(x+y+z) - omega t), rho = d_t u (reading S17); period L = 2 per axis."""
    x, y, z = w.centres(level, ibox)
    ph = PLANE_K * (z[:, None, None] + y[None, :, None] + x[None, None, :]) - PLANE_OMEGA * t
    return np.sin(ph) if comp < w.nfields else -PLANE_OMEGA * np.cos(ph)


def plane_wave_init(w: Workload, level: int, ibox: int, comp: int) -> np.ndarray:
    return plane_wave_exact(w, level, ibox, comp, 0.0)


def quadratic_exact(w: Workload, level: int, ibox: int, comp: int, t: float, pad: int = 0) -> np.ndarray:
    """u = x^2 + y^2 + z^2 + 3 t^2, rho = 6 t: an exact solution of the wave equation (u_tt = 6 = Lap u) that
    every operator of the scheme reproduces exactly (away from the periodic seam of level 0)."""
    x, y, z = w.centres(level, ibox, pad)
    if comp < w.nfields:
        return z[:, None, None] ** 2 + y[None, :, None] ** 2 + x[None, None, :] ** 2 + 3.0 * t * t
    return np.full((len(z), len(y), len(x)), 6.0 * t)


def quadratic_init(w: Workload, level: int, ibox: int, comp: int) -> np.ndarray:
    return quadratic_exact(w, level, ibox, comp, 0.0)


def multi_gaussian_init(ngauss: int = 8):
    """u_f = sum_m a exp(-|x-c|^2/(2 w^2)), a~U(-1,1), c~U(-.5,.5)^3, w~U(.05,.3); rho_f = 0 (S23)."""
    def f(w: Workload, level: int, ibox: int, comp: int) -> np.ndarray:
        b = w.box(level, ibox)
        v = np.zeros((b.n[2], b.n[1], b.n[0]))
        if comp >= w.nfields:
            return v
        m = np.arange(ngauss, dtype=np.uint64)
        a = 2.0 * counter_uniform01(SEED, [1000, comp, 0], m) - 1.0
        cx = counter_uniform01(SEED, [1000, comp, 1], m) - 0.5
        cy = counter_uniform01(SEED, [1000, comp, 2], m) - 0.5
        cz = counter_uniform01(SEED, [1000, comp, 3], m) - 0.5
        wd = 0.05 + 0.25 * counter_uniform01(SEED, [1000, comp, 4], m)
        x, y, z = w.centres(level, ibox)
        for i in range(ngauss):
            # separable: exp(-(dx^2+dy^2+dz^2)/(2w^2)) = ex*ey*ez
            s = 1.0 / (2.0 * wd[i] ** 2)
            ex = np.exp(-s * (x - cx[i]) ** 2)
            ey = np.exp(-s * (y - cy[i]) ** 2)
            ez = np.exp(-s * (z - cz[i]) ** 2)
            v += a[i] * ez[:, None, None] * ey[None, :, None] * ex[None, None, :]
        return v
    return f


def coupling_matrix(nfields: int, seed: int = SEED) -> np.ndarray:
    """Symmetric negative-semidefinite A (reading S21): G_ij ~ N(0, var 0.01); S = (G+G^T)/2;
    A = S - max_i sum_j |S_ij| * I (Gershgorin shift)."""
    cnt = np.arange(nfields * nfields, dtype=np.uint64)
    G = 0.1 * counter_normal(seed, [2000], cnt).reshape(nfields, nfields)
    S = 0.5 * (G + G.T)
    shift = np.max(np.sum(np.abs(S), axis=1))
    return np.ascontiguousarray(S - shift * np.eye(nfields))


# ----------------------------------------------------------------------------------------------
# the five BASELINE.json configurations (+ scaled-down variants for tests)
# ----------------------------------------------------------------------------------------------
def cfg1() -> Workload:
    return Workload("cfg1: scalar wave, 2 levels x 32^3, Gaussian exp(-r^2/0.1) + 1e-6 noise",
                    nested_cubes(2, 32), (32, 32, 32), coarse_steps=8, init=gaussian_init(0.1))


def cfg2(n: int = 32) -> Workload:
    w = Workload(f"cfg2: convergence ladder rung, 2 levels x {n}^3, plane wave",
                 nested_cubes(2, n), (n, n, n), init=plane_wave_init)
    w.coarse_steps = int(round(1.0 / w.dt_coarse))  # to t = 1: 64 / 128 / 256
    return w


def cfg3(n: int = 128, nlevels: int = 4) -> Workload:
    return Workload(f"cfg3: scalar wave, {nlevels} levels x {n}^3, Gaussian w=0.05 + 1e-6 noise",
                    nested_cubes(nlevels, n), (n, n, n), coarse_steps=50,
                    init=gaussian_init(2 * 0.05 ** 2))


def cfg4(n: int = 96, nlevels: int = 7, nfields: int = 22) -> Workload:
    """BBH-shaped: nlevels-1 centred n^3 levels + a finest level of two boxes (reading S20: for n = 96
    the boxes are 80x96x96, parent-local x in [4,44) and [52,92), y,z in [24,72))."""
    boxes = nested_cubes(nlevels - 1, n)
    p = boxes[-1]
    h, q = n // 2, n // 4
    nxp = h - 8  # parent cells per box in x: margin 4 each side, gap 8
    for x0 in (4, h + 4):
        boxes.append(Box(nlevels - 1,
                         (2 * (p.lo[0] + x0), 2 * (p.lo[1] + q), 2 * (p.lo[2] + q)),
                         (2 * nxp, 2 * h, 2 * h)))
    return Workload(f"cfg4: BBH-shaped, {nlevels} levels x {n}^3 (finest: 2 boxes), F={nfields}",
                    boxes, (n, n, n), nfields=nfields, coupling=coupling_matrix(nfields),
                    coarse_steps=20, init=multi_gaussian_init(8),
                    note="S20: finest level = two (n-16) x n x n boxes")


def cfg5(n: int = 256, nlevels: int = 6) -> Workload:
    return Workload(f"cfg5: scalar wave, {nlevels} levels x {n}^3, Gaussian w=0.05 + 1e-6 noise",
                    nested_cubes(nlevels, n), (n, n, n), coarse_steps=20,
                    init=gaussian_init(2 * 0.05 ** 2))


def cfg5_spacings(n: int = 64, nlevels: int = 6) -> Workload:
    """cfg 5's finest grid spacing (2 / 8192) and its spacing ratio between levels, on `nlevels` nested n^3 boxes: the
    domain shrinks instead of the resolution. With nlevels = 6 every level has cfg 5's dx and dt and the finest level
    cfg 5's 128 RHS evaluations per coarse step — the rounding behaviour of the full configuration at a size the oracle
    steps in seconds (S27). The pulse is cfg 5's (periodic images overlap a little at the small domain's
    edge: irrelevant to what this input is for)."""
    half = n * 2.0 ** (nlevels - 1) / 8192.0
    return Workload(f"cfg5 spacings (dx_finest = 2/8192), {nlevels} levels x {n}^3", nested_cubes(nlevels, n), (n, n, n),
                    xlo=(-half,) * 3, xhi=(half,) * 3, coarse_steps=1, init=gaussian_init(2 * 0.05 ** 2))


def ragged_small() -> Workload:
    """Test-only: non-cubic, odd-tile sizes, off-centre child, two grandchildren; F = 2 with coupling."""
    boxes = [Box(0, (0, 0, 0), (40, 24, 28)),
             Box(1, (10, 8, 12), (44, 28, 26)),
             Box(2, (30, 26, 34), (24, 18, 20)),
             Box(2, (66, 24, 34), (22, 20, 18))]
    return Workload("ragged: 3 levels, non-cubic boxes, 2 fields coupled", boxes, (40, 24, 28),
                    nfields=2, coupling=coupling_matrix(2), coarse_steps=2,
                    xlo=(-1.0, -0.6, -0.7), xhi=(1.0, 0.6, 0.7),
                    init=multi_gaussian_init(3))


def global_index_init(w: Workload, level: int, ibox: int, comp: int) -> np.ndarray:
    """Smooth pulse + a ripple that depends on the LEVEL-GLOBAL cell index only: every decomposition of a level
    into boxes gets the same numbers (test data of the same-level ghost exchange)."""
    b = w.box(level, ibox)
    x, y, z = w.centres(level, ibox)
    i, j, k = (np.arange(b.lo[a], b.lo[a] + b.n[a], dtype=np.float64) for a in range(3))
    r2 = z[:, None, None] ** 2 + y[None, :, None] ** 2 + (x[None, None, :] - 0.1) ** 2
    rip = np.sin(12.9898 * i[None, None, :] + 78.233 * j[None, :, None] + 37.719 * k[:, None, None] + comp + level)
    amp = 1.0 if comp < w.nfields else 0.3
    return amp * np.exp(-r2 / 0.1) + 1e-3 * rip


def sibling_cut(cuts_x=(), cuts_y=(), cuts_z=(), nfields: int = 1, ko_sigma: float = 0.0,
                near: bool = False) -> Workload:
    """Test-only: 3 levels; level 1 = the region [12, 36)^3 of a 24^3 level 0, cut into abutting boxes at the given
    level-global indices (no cuts = one box); level 2 = one 8x12x16 box that nests in a piece of every cut with
    x in {24}, y in {20, 22}, z in {20}. `near` adds a level-1 box two cells away from the cut region (only part
    of its ghost shell lies inside a sibling)."""
    lo, n = 12, 24

    def segs(cuts):
        e = [lo] + list(cuts) + [lo + n]
        return list(zip(e[:-1], e[1:]))
    boxes = [Box(0, (0, 0, 0), (32, 24, 24))]
    for z0, z1 in segs(cuts_z):
        for y0, y1 in segs(cuts_y):
            for x0, x1 in segs(cuts_x):
                boxes.append(Box(1, (x0, y0, z0), (x1 - x0, y1 - y0, z1 - z0)))
    if near:
        boxes.append(Box(1, (38, 14, 16), (14, 18, 12)))
    boxes.append(Box(2, (56, 52, 48), (8, 12, 16)))
    return Workload("siblings: level 1 cut into %d boxes" % (len(boxes) - 2), boxes, (32, 24, 24), nfields=nfields,
                    coupling=coupling_matrix(nfields) if nfields > 1 else None, coarse_steps=2,
                    xlo=(-4.0 / 3.0, -1.0, -1.0), xhi=(4.0 / 3.0, 1.0, 1.0),
                    init=global_index_init, ko_sigma=ko_sigma)


def cut_finest(w: Workload, pieces: int, axis: int = 2) -> Workload:
    """The same hierarchy with every box of the finest level cut into `pieces` abutting slabs along `axis`
    (same cells, same work; the slabs exchange ghosts — NEXT-2). Measurement variant of a BASELINE configuration."""
    top = w.nlevels - 1
    boxes = [b for b in w.boxes if b.level != top]
    for b in w.level_boxes(top):
        step = (b.n[axis] // pieces) & ~1
        assert step >= 8
        for p in range(pieces):
            lo, n = list(b.lo), list(b.n)
            lo[axis] = b.lo[axis] + p * step
            n[axis] = step if p < pieces - 1 else b.n[axis] - p * step
            boxes.append(Box(top, tuple(lo), tuple(n)))
    out = dataclasses.replace(w, boxes=boxes)
    out.name = w.name + f", finest level cut into {pieces} abutting slabs"
    return out


# ----------------------------------------------------------------------------------------------
# the paper's own scalar-wave test (eqs 41-42, Fig. 1)
# ----------------------------------------------------------------------------------------------
SPH_A, SPH_SIGMA = 1.0, 0.25 / math.sqrt(2.0)


def spherical_wave_exact(w: Workload, level: int, ibox: int, comp: int, t: float, sigma: float = None) -> np.ndarray:
    """u = [f(t-r) - f(t+r)] / r,  Pi = -[f(t-r)(t-r) - f(t+r)(t+r)] / (sigma^2 r),  f(v) = A exp(-v^2 / (2 sigma^2)),
    A = 1, sigma = 0.25/sqrt(2) (eqs 41-42). Cell-centred grids never put a centre at r = 0 (S1)."""
    sg = SPH_SIGMA if sigma is None else sigma
    x, y, z = w.centres(level, ibox)
    r = np.sqrt(z[:, None, None] ** 2 + y[None, :, None] ** 2 + x[None, None, :] ** 2)
    f = lambda v: SPH_A * np.exp(-v * v / (2.0 * sg ** 2))  # noqa: E731
    if comp < w.nfields:
        return (f(t - r) - f(t + r)) / r
    return -(f(t - r) * (t - r) - f(t + r) * (t + r)) / (sg ** 2 * r)


def paper_wave(n0: int = 64) -> Workload:
    """The paper's Fig. 1 set-up: three levels with refinement boundaries at r = 4, 1, 0.5 (read as
    the half-widths of cubic boxes), dx_0 = 8 / n0: n0 = 64, 96, 128 are its h_1 = 1/8, h_1/1.5, h_1/2. The outer
    boundary is periodic here (S9): valid until the pulse reaches r = 4."""
    assert n0 % 16 == 0
    q = n0 // 4
    boxes = [Box(0, (0, 0, 0), (n0, n0, n0)), Box(1, (n0 - q,) * 3, (2 * q,) * 3), Box(2, (2 * n0 - q,) * 3, (2 * q,) * 3)]
    return Workload(f"paper Fig. 1: Gaussian spherical wave, 3 levels (r = 4, 1, 0.5), dx_0 = 8/{n0}", boxes,
                    (n0, n0, n0), xlo=(-4.0, -4.0, -4.0), xhi=(4.0, 4.0, 4.0),
                    init=lambda w, l, ib, c: spherical_wave_exact(w, l, ib, c, 0.0))
