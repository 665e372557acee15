"""Pins for the oracle's spatial operators, index maps and the whole scheme. CPU only.

What fixes the expected values: the rational weights (tests/golden/interp_weights.txt), polynomial
exactness, geometry (cell-centre coordinates), the closed-form amplification matrix of RK4 + the
4th-order Laplacian on a Fourier mode, the exact plane-wave solution (reading S17), linearity."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from paper_2503_09629_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    for l in open(os.path.join(GOLD, "interp_weights.txt")):
        t = l.split()
        if t and t[0] == name:
            return np.array([float(Fraction(x)) for x in t[1:]])
    raise KeyError(name)


def _poly(x, y, z, cx, cy, cz):
    """Tensor polynomial sum_a cx[a] x^a * sum_b cy[b] y^b * sum_c cz[c] z^c on a [z][y][x] grid."""
    px = sum(c * x ** a for a, c in enumerate(cx))
    py = sum(c * y ** a for a, c in enumerate(cy))
    pz = sum(c * z ** a for a, c in enumerate(cz))
    return pz[:, None, None] * py[None, :, None] * px[None, None, :]


# ----------------------------------------------------------------------------------------------
def test_weights_match_rationals(oracle_mod):
    o = oracle_mod
    w1 = _gold("prolong1")
    assert np.allclose(o.prolong_weights(1), w1, rtol=0, atol=2e-16)
    assert np.allclose(o.prolong_weights(0), w1[::-1], rtol=0, atol=2e-16)  # mirror symmetry
    assert np.allclose(o.restrict_weights(), _gold("restrict"), rtol=0, atol=2e-16)
    assert abs(o.prolong_weights(0).sum() - 1) < 1e-15 and abs(o.restrict_weights().sum() - 1) < 1e-15


def test_weights_polynomial_exactness(oracle_mod):
    o = oracle_mod
    nodes5 = np.arange(-2.0, 3.0)
    for par, x in ((0, -0.25), (1, 0.25)):
        w = o.prolong_weights(par)
        for p in range(5):
            assert abs(w @ nodes5 ** p - x ** p) < 1e-14
        assert abs(w @ nodes5 ** 5 - x ** 5) > 1e-3  # and not of higher degree
    nodes6 = np.arange(-2.5, 3.0)
    r = o.restrict_weights()
    for p in range(6):
        assert abs(r @ nodes6 ** p - (1.0 if p == 0 else 0.0)) < 1e-13
    assert abs(r @ nodes6 ** 6) > 1e-3


# ----------------------------------------------------------------------------------------------
def _two_level(n=16, F=1):
    return wl.Workload("t", wl.nested_cubes(2, n), (n, n, n), nfields=F)


def test_laplacian_polynomial_exactness_and_rhs_structure(oracle_mod):
    """k_1 = f(y_n): k_u = rho, k_rho = Lap u exact for polynomials of degree <= 5 per axis, away from
    the periodic seam."""
    w = wl.Workload("t", [wl.Box(0, (0, 0, 0), (12, 10, 14))], (12, 10, 14),
                    xlo=(-0.6, -0.5, -0.7), xhi=(0.6, 0.5, 0.7))
    H = oracle_mod.OracleHierarchy(w.boxes, w.domain_cells, 1, 3, w.xlo, w.xhi)
    x, y, z = w.centres(0, 0)
    cx, cy, cz = [1, -2, .5, 3, -1, 2], [.3, 1, -1, .5, 2, -3], [2, .1, -.7, 1, 1, .4]
    u = _poly(x, y, z, cx, cy, cz)
    rho = _poly(x, y, z, [1, 1], [2, -1], [0.5, 3])
    H.set_state(0, 0, 0, u)
    H.set_state(0, 0, 1, rho)
    H.step(1e-9, True)
    k1u = H.read(0, 0, 0, slot=2)
    k1r = H.read(0, 0, 1, slot=2)
    assert np.array_equal(k1u, rho)

    def d2(c):
        return [c[a] * a * (a - 1) for a in range(2, len(c))]

    lap = _poly(x, y, z, d2(cx), cy, cz) + _poly(x, y, z, cx, d2(cy), cz) + _poly(x, y, z, cx, cy, d2(cz))
    s = (slice(2, -2),) * 3
    assert np.max(np.abs(k1r[s] - lap[s])) < 2e-10 * np.max(np.abs(lap))


@pytest.mark.parametrize("sub", [True, False])
def test_prolongation_and_restriction_exact_for_quartics(oracle_mod, sub):
    """Whole-hierarchy check of the index maps + operators: for u = tensor quartic (rho = 0) and a
    vanishing step, the child's ghosts must equal the polynomial at the ghost cell centres and the
    restricted parent cells must equal it at the parent centres."""
    w = wl.ragged_small()
    H = oracle_mod.OracleHierarchy(w.boxes, w.domain_cells, w.nfields, w.ghost, w.xlo, w.xhi, None)
    cx, cy, cz = [1, -2, .5, 3, -1], [.3, 1, -1, .5, 2], [2, .1, -.7, 1, 1]
    for l in range(w.nlevels):
        for ib in range(len(w.level_boxes(l))):
            x, y, z = w.centres(l, ib)
            H.set_state(l, ib, 0, _poly(x, y, z, cx, cy, cz))
            H.set_state(l, ib, 1, _poly(x, y, z, cz, cx, cy))
    H.step(1e-10, sub)
    scale = 10.0
    for l in range(1, w.nlevels):
        for ib in range(len(w.level_boxes(l))):
            x, y, z = w.centres(l, ib, pad=w.ghost)
            for comp, cc in ((0, (cx, cy, cz)), (1, (cz, cx, cy))):
                got = H.read(l, ib, comp, padded=True)
                assert np.max(np.abs(got - _poly(x, y, z, *cc))) < 1e-9 * scale, (l, ib, comp)
    # restriction: parent cells under the children (level 0 is not periodic-polynomial near its seam,
    # but the covered cells are far from it)
    b1 = w.box(1, 0)
    x, y, z = w.centres(0, 0)
    got = H.read(0, 0, 0)
    want = _poly(x, y, z, cx, cy, cz)
    sl = tuple(slice(b1.lo[a] // 2, (b1.lo[a] + b1.n[a]) // 2) for a in (2, 1, 0))
    assert np.max(np.abs(got[sl] - want[sl])) < 1e-9 * scale


def test_ghost_index_map_brute_force_geometry(oracle_mod):
    """(I>>1, I&1) against floating-point geometry: the containing parent cell is the one whose centre
    is exactly dx_p/4 away on every axis; parity 1 = fine centre on the + side."""
    w = wl.ragged_small()
    H = oracle_mod.OracleHierarchy(w.boxes, w.domain_cells, w.nfields, w.ghost, w.xlo, w.xhi, None)
    g = w.ghost
    for l in (1, 2):
        for ib in range(len(w.level_boxes(l))):
            b = w.box(l, ib)
            gm = H.ghost_map(l, ib)
            nshell = np.prod([n + 2 * g for n in b.n]) - np.prod(b.n)
            assert gm.shape == (nshell, 7)
            # canonical order: k, j, i ascending, interior skipped
            order = [(k, j, i) for k in range(-g, b.n[2] + g) for j in range(-g, b.n[1] + g)
                     for i in range(-g, b.n[0] + g)
                     if not (0 <= i < b.n[0] and 0 <= j < b.n[1] and 0 <= k < b.n[2])]
            assert np.array_equal(gm[:, [2, 1, 0]], np.array(order, dtype=np.int32))
            # find the parent box by geometry
            parents = w.level_boxes(l - 1)
            for a in range(3):
                dxf = (w.xhi[a] - w.xlo[a]) / (w.domain_cells[a] * 2 ** l)
                dxp = 2 * dxf
                xf = w.xlo[a] + (b.lo[a] + gm[:, a] + 0.5) * dxf
                ok_any = np.zeros(len(gm), dtype=bool)
                for p in parents:
                    xp = w.xlo[a] + (p.lo[a] + gm[:, 3 + a] + 0.5) * dxp
                    par = (gm[:, 6] >> a) & 1
                    ok = np.abs((xf - xp) - np.where(par == 1, 0.25, -0.25) * dxp) < 1e-12 * dxp
                    ok_any |= ok
                assert ok_any.all()
            # footprint stays inside the parent's interior
            pidx = gm[:, 3:6]
            assert pidx.min() >= 2


def test_ghost_map_negative_indices_floor(oracle_mod):
    """A box at global index 8 on level 1 with ghost cells reaching index 5: parents floor correctly.
    (Negative global indices cannot occur under the nesting rule; the floor is still exercised for odd
    indices below lo.)"""
    boxes = [wl.Box(0, (0, 0, 0), (16, 16, 16)), wl.Box(1, (8, 8, 8), (16, 16, 16))]
    H = oracle_mod.OracleHierarchy(boxes, (16, 16, 16))
    gm = H.ghost_map(1, 0)
    first = gm[0]
    assert list(first[:3]) == [-3, -3, -3]
    assert list(first[3:6]) == [2, 2, 2] and first[6] == 7  # global 5 -> parent 2, parity 1


# ----------------------------------------------------------------------------------------------
def _amp_matrix(kappa2, dt):
    M = np.array([[0.0, 1.0], [-kappa2, 0.0]])
    Z = dt * M
    return np.eye(2) + Z + Z @ Z / 2 + Z @ Z @ Z / 6 + Z @ Z @ Z @ Z / 24


def test_single_level_closed_form_amplification(oracle_mod):
    """One periodic level, data on Fourier modes: after n steps (a, b) -> R(dt M)^n (a, b) with
    M = [[0,1],[-kappa^2,0]], kappa^2 = sum_axis (30 - 32 cos(k h) + 2 cos(2 k h))/(12 h^2)."""
    n = 16
    w = wl.Workload("t", [wl.Box(0, (0, 0, 0), (n, n, n))], (n, n, n))
    H = oracle_mod.OracleHierarchy(w.boxes, w.domain_cells)
    x, y, z = w.centres(0, 0)
    kv = math.pi * np.array([1, 2, -1])  # integer multiples of 2 pi / L, L = 2
    ph = kv[2] * z[:, None, None] + kv[1] * y[None, :, None] + kv[0] * x[None, None, :]
    s, c = np.sin(ph), np.cos(ph)
    H.set_state(0, 0, 0, 0.7 * s - 0.2 * c)
    H.set_state(0, 0, 1, 1.1 * s + 0.4 * c)
    h = w.dx(0)
    kappa2 = sum((30 - 32 * math.cos(k * h) + 2 * math.cos(2 * k * h)) / (12 * h * h) for k in kv)
    dt, nsteps = 0.25 * h, 40
    R = np.linalg.matrix_power(_amp_matrix(kappa2, dt), nsteps)
    for _ in range(nsteps):
        H.step(dt, True)
    a, b = R @ np.array([0.7, 1.1])
    cc, d = R @ np.array([-0.2, 0.4])
    assert np.max(np.abs(H.read_level(0, 0, 0) - (a * s + cc * c))) < 2e-13
    assert np.max(np.abs(H.read_level(0, 0, 1) - (b * s + d * c))) < 2e-12
    assert abs(H.time - nsteps * dt) < 1e-15


def test_coupled_system_closed_form(oracle_mod):
    """With coupling A and data along an eigenvector of A (eigenvalue lam <= 0): kappa^2 -> kappa^2 - lam."""
    n, F = 12, 3
    A = wl.coupling_matrix(F)
    lam, vec = np.linalg.eigh(A)
    assert lam.max() <= 1e-12 and np.allclose(A, A.T)
    w = wl.Workload("t", [wl.Box(0, (0, 0, 0), (n, n, n))], (n, n, n), nfields=F, coupling=A)
    H = oracle_mod.OracleHierarchy(w.boxes, w.domain_cells, F, 3, w.xlo, w.xhi, A)
    x, y, z = w.centres(0, 0)
    kv = math.pi * np.array([1, 0, 1])
    s = np.sin(kv[2] * z[:, None, None] + kv[1] * y[None, :, None] + kv[0] * x[None, None, :])
    e = vec[:, 1]
    for f in range(F):
        H.set_state(0, 0, f, e[f] * s)
        H.set_state(0, 0, F + f, -0.5 * e[f] * s)
    h = w.dx(0)
    kappa2 = sum((30 - 32 * math.cos(k * h) + 2 * math.cos(2 * k * h)) / (12 * h * h) for k in kv) - lam[1]
    dt, nsteps = 0.25 * h, 10
    for _ in range(nsteps):
        H.step(dt, False)
    a, b = np.linalg.matrix_power(_amp_matrix(kappa2, dt), nsteps) @ np.array([1.0, -0.5])
    for f in range(F):
        assert np.max(np.abs(H.read_level(0, 0, f) - a * e[f] * s)) < 1e-13
        assert np.max(np.abs(H.read_level(0, 0, F + f) - b * e[f] * s)) < 1e-12


def test_single_level_pde_accuracy(oracle_mod):
    """Error vs the exact plane wave ~ omega T [(k h)^4/180 * ... ]: SURVEY quotes 5.13e-5 measured by an
    independent prototype at 32^3, t = 1 (leading-term estimate 4.73e-5)."""
    n = 32
    w = wl.Workload("t", [wl.Box(0, (0, 0, 0), (n, n, n))], (n, n, n), init=wl.plane_wave_init)
    H = oracle_mod.OracleHierarchy.from_workload(w)
    nsteps = int(round(1.0 / w.dt_coarse))
    for _ in range(nsteps):
        H.step(w.dt_coarse, True)
    err = np.max(np.abs(H.read_level(0, 0, 0) - wl.plane_wave_exact(w, 0, 0, 0, 1.0)))
    assert 4.6e-5 < err < 5.6e-5, err


# ----------------------------------------------------------------------------------------------
def _run(oracle_mod, w, nsteps, sub, scale=None):
    H = oracle_mod.OracleHierarchy(w.boxes, w.domain_cells, w.nfields, w.ghost, w.xlo, w.xhi, w.coupling)
    for l in range(w.nlevels):
        for ib in range(len(w.level_boxes(l))):
            for c in range(w.ncomp):
                a = w.initial_state(l, ib, c)
                H.set_state(l, ib, c, a if scale is None else scale(l, ib, c, a))
    for _ in range(nsteps):
        H.step(w.dt_coarse, sub)
    return H


@pytest.mark.parametrize("sub", [True, False])
def test_linearity_and_constant_fixed_point(oracle_mod, sub):
    w1 = wl.ragged_small()
    w2 = wl.ragged_small()
    w2.init = wl.gaussian_init(0.08, noise=1e-3)
    al, be = 0.75, -1.5

    def combo(l, ib, c, a):
        return al * a + be * w2.initial_state(l, ib, c)

    Ha, Hb, Hc = _run(oracle_mod, w1, 2, sub), _run(oracle_mod, w2, 2, sub), _run(oracle_mod, w1, 2, sub, combo)
    for l in range(w1.nlevels):
        for ib in range(len(w1.level_boxes(l))):
            for c in range(w1.ncomp):
                lin = al * Ha.read_level(l, ib, c) + be * Hb.read_level(l, ib, c)
                assert np.max(np.abs(Hc.read_level(l, ib, c) - lin)) < 1e-12
    # constant u, zero rho, no coupling: fixed point to rounding
    w3 = wl.ragged_small()
    w3.coupling = None
    w3.init = lambda w, l, ib, c: np.full((w.box(l, ib).n[2], w.box(l, ib).n[1], w.box(l, ib).n[0]),
                                          1.0 if c < w.nfields else 0.0)
    Hk = _run(oracle_mod, w3, 2, sub)
    for l in range(w3.nlevels):
        for ib in range(len(w3.level_boxes(l))):
            assert np.max(np.abs(Hk.read_level(l, ib, 0) - 1.0)) < 1e-13
            assert np.max(np.abs(Hk.read_level(l, ib, 2))) < 1e-9  # rho: rounding of Lap(1) * dt


def test_octahedral_symmetry_preserved(oracle_mod):
    """Noise-free centred Gaussian on nested cubes: the solution stays symmetric under x <-> y <-> z
    permutations and reflections to rounding (catches transposed axes / parity mix-ups)."""
    w = wl.Workload("t", wl.nested_cubes(3, 16), (16, 16, 16), init=wl.gaussian_init(0.1, noise=0.0))
    H = _run(oracle_mod, w, 3, True)
    for l in range(3):
        for c in range(2):
            a = H.read_level(l, 0, c)
            for b in (a.transpose(1, 0, 2), a.transpose(0, 2, 1), a[::-1], a[:, ::-1], a[:, :, ::-1]):
                assert np.max(np.abs(a - b)) < 1e-13


# ----------------------------------------------------------------------------------------------
def _ladder_errors(oracle_mod, n, sub):
    w = wl.cfg2(n)
    H = oracle_mod.OracleHierarchy.from_workload(w)
    for _ in range(w.coarse_steps):
        H.step(w.dt_coarse, sub)
    assert abs(H.time - 1.0) < 1e-12
    errs = [np.max(np.abs(H.read_level(l, 0, 0) - wl.plane_wave_exact(w, l, 0, 0, 1.0))) for l in (0, 1)]
    return errs, [H.read_level(l, 0, 0) for l in (0, 1)]


@pytest.mark.slow
def test_convergence_ladder_and_sub_vs_uniform(oracle_mod):
    """BASELINE config 2 / PAPER.md:238,246: 4th-order convergence against the exact plane wave, with and
    without subcycling; the two modes agree to truncation level. Indicative numbers from SURVEY.md
    Appendix B (independent numpy prototype): 32^3: 6.20e-5 / 6.21e-5 (sub), 6.00e-5 / 6.01e-5 (uniform),
    |sub - uniform| 5.5e-6; 64^3: 3.97e-6 / 3.98e-6 (sub), 3.83e-6 / 3.84e-6, |diff| 6.5e-7."""
    e32s, u32s = _ladder_errors(oracle_mod, 32, True)
    e64s, u64s = _ladder_errors(oracle_mod, 64, True)
    e32u, u32u = _ladder_errors(oracle_mod, 32, False)
    e64u, u64u = _ladder_errors(oracle_mod, 64, False)
    for e32, e64 in ((e32s, e64s), (e32u, e64u)):
        for l in (0, 1):
            order = math.log2(e32[l] / e64[l])
            assert 3.8 < order < 4.2, (l, e32, e64, order)
    assert np.allclose(e32s, [6.201e-5, 6.208e-5], rtol=2e-3)
    assert np.allclose(e64s, [3.972e-6, 3.984e-6], rtol=2e-3)
    assert np.allclose(e32u, [6.001e-5, 6.009e-5], rtol=2e-3)
    assert np.allclose(e64u, [3.829e-6, 3.838e-6], rtol=2e-3)
    d32 = max(np.max(np.abs(a - b)) for a, b in zip(u32s, u32u))
    d64 = max(np.max(np.abs(a - b)) for a, b in zip(u64s, u64u))
    assert d32 < 0.2 * max(e32s) and d64 < 0.3 * max(e64s)
    assert 2.5 < math.log2(d32 / d64) < 3.6  # the difference itself converges at ~3rd order (S12)


@pytest.mark.parametrize("sub", [True, False])
def test_composite_scheme_exact_for_quadratic_solution(oracle_mod, sub):
    """Pins the COMPOSITE multi-level scheme to a closed form: u = x^2+y^2+z^2+3t^2, rho = 6t solves the wave
    equation, the 4th-order Laplacian, the quartic prolongation and the quintic restriction are exact on it,
    RK4 is exact for solutions quadratic in t, and so are eq (10) and the stage formulas (15)-(18) for a linear
    autonomous system (d3y/dt3 = f_y d2y/dt2 and 4 (k_3 - k_2) / h_p^2 = f_y d2y/dt2 hold exactly; with the
    child's h in place of the parent's, S5, the h^3 terms would not cancel). One coarse step of a 3-level
    hierarchy (2 and 4 subcycled fine steps, theta = 0 and 1/2 fills, both restrictions) must therefore
    reproduce the polynomial to rounding wherever the periodic seam of level 0 (8 cells per step) has not reached."""
    n = 64
    w = wl.Workload("quadratic", wl.nested_cubes(3, n), (n, n, n), init=wl.quadratic_init)
    H = oracle_mod.OracleHierarchy.from_workload(w)
    H.step(w.dt_coarse, sub)
    t = w.dt_coarse
    for l in (1, 2):
        for c in (0, 1):
            got = H.read(l, 0, c, padded=True)
            want = wl.quadratic_exact(w, l, 0, c, t, pad=w.ghost)
            assert np.max(np.abs(got - want)) < 2e-12, (sub, l, c, float(np.max(np.abs(got - want))))
    m = slice(10, n - 10)
    for c in (0, 1):
        got = H.read(0, 0, c)[m, m, m]
        want = wl.quadratic_exact(w, 0, 0, c, t)[m, m, m]
        assert np.max(np.abs(got - want)) < 2e-12, (sub, 0, c)


def test_kreiss_oliger_closed_form_amplification(oracle_mod):
    """Eqs (35)-(36) on one periodic level: on a Fourier mode Q acts as the number
    q = sigma/64 sum_axis (2 cos 3kh - 12 cos 2kh + 30 cos kh - 20)/h  (<= 0: dissipative), on u AND rho, so
    M = [[q, 1], [-kappa^2, q]] and n steps apply R(dt M)^n. A wrong sign, a dropped variable, a wrong power of h
    or a transposed stencil weight changes q."""
    n, sigma = 16, 0.3
    w = wl.Workload("t", [wl.Box(0, (0, 0, 0), (n, n, n))], (n, n, n), ko_sigma=sigma)
    H = oracle_mod.OracleHierarchy.from_workload(
        wl.Workload("t", w.boxes, w.domain_cells, ko_sigma=sigma, init=lambda *a: np.zeros((n, n, n))))
    x, y, z = w.centres(0, 0)
    kv = math.pi * np.array([3, -2, 5])
    ph = kv[2] * z[:, None, None] + kv[1] * y[None, :, None] + kv[0] * x[None, None, :]
    s, c = np.sin(ph), np.cos(ph)
    H.set_state(0, 0, 0, 0.7 * s - 0.2 * c)
    H.set_state(0, 0, 1, 1.1 * s + 0.4 * c)
    h = w.dx(0)
    kappa2 = sum((30 - 32 * math.cos(k * h) + 2 * math.cos(2 * k * h)) / (12 * h * h) for k in kv)
    q = sigma / 64.0 * sum((2 * math.cos(3 * k * h) - 12 * math.cos(2 * k * h) + 30 * math.cos(k * h) - 20) / h for k in kv)
    assert q < 0
    dt, nsteps = 0.25 * h, 25
    Z = dt * np.array([[q, 1.0], [-kappa2, q]])
    R = np.linalg.matrix_power(np.eye(2) + Z + Z @ Z / 2 + Z @ Z @ Z / 6 + Z @ Z @ Z @ Z / 24, nsteps)
    for _ in range(nsteps):
        H.step(dt, True)
    a, b = R @ np.array([0.7, 1.1])
    cc, d = R @ np.array([-0.2, 0.4])
    assert np.max(np.abs(H.read_level(0, 0, 0) - (a * s + cc * c))) < 2e-13
    assert np.max(np.abs(H.read_level(0, 0, 1) - (b * s + d * c))) < 2e-12
    # the undamped scheme gives a different answer at this mode by far more than the tolerance
    R0 = np.linalg.matrix_power(_amp_matrix(kappa2, dt), nsteps)
    assert abs((R0 @ np.array([0.7, 1.1]))[0] - a) > 1e-3


@pytest.mark.parametrize("sub", [True, False])
def test_composite_scheme_with_dissipation_exact_for_quadratic_solution(oracle_mod, sub):
    """Q annihilates polynomials of degree <= 5, so the exact quadratic solution must survive the composite
    3-level step with dissipation switched on exactly as without it (every ghost layer the 7-point stencil
    reads, at every stage, must hold the polynomial)."""
    n = 64
    w = wl.Workload("quadratic+KO", wl.nested_cubes(3, n), (n, n, n), init=wl.quadratic_init, ko_sigma=0.2)
    H = oracle_mod.OracleHierarchy.from_workload(w)
    H.step(w.dt_coarse, sub)
    t = w.dt_coarse
    for l in (1, 2):
        for c in (0, 1):
            got = H.read(l, 0, c, padded=True)
            assert np.max(np.abs(got - wl.quadratic_exact(w, l, 0, c, t, pad=w.ghost))) < 5e-12, (sub, l, c)
    m = slice(14, n - 14)  # the seam now travels 3 cells per stage
    for c in (0, 1):
        assert np.max(np.abs(H.read(0, 0, c)[m, m, m] - wl.quadratic_exact(w, 0, 0, c, t)[m, m, m])) < 5e-12


def test_dissipation_damps_grid_noise_and_keeps_smooth_data(oracle_mod):
    """Nyquist-scale noise decays under Q (one level: |amplification| < 1 for the highest mode), while a smooth
    mode changes by O(h^5)."""
    n = 16
    box = [wl.Box(0, (0, 0, 0), (n, n, n))]
    i = np.arange(n)
    checker = ((-1.0) ** (i[:, None, None] + i[None, :, None] + i[None, None, :]))
    out = {}
    for sigma in (0.0, 0.5):
        H = oracle_mod.OracleHierarchy(box, (n, n, n), ko_sigma=sigma)
        H.set_state(0, 0, 0, np.zeros((n, n, n)))
        H.set_state(0, 0, 1, 1e-3 * checker)      # rho at the Nyquist mode: Lap u = 0 keeps u = t * rho only
        for _ in range(10):
            H.step(0.25 * 2.0 / n, True)
        out[sigma] = np.max(np.abs(H.read_level(0, 0, 1)))
    assert out[0.5] < 0.2 * out[0.0]


@pytest.mark.slow
def test_paper_fig1_spherical_wave_fourth_order(oracle_mod):
    """The paper's own validation (eqs 41-42, Fig. 1): Gaussian spherical wave, three levels with
    refinement boundaries at r = 4, 1, 0.5, resolutions h_1 = 1/8, h_1/1.5, h_1/2; errors on the second refinement
    level against the exact solution after the pulse has crossed the level-2 boundary (t = 0.75), 'assuming
    fourth-order convergence' for subcycling and for uniform stepping alike."""
    T = 0.75
    err = {}
    for sub, n0 in ((True, 64), (True, 96), (True, 128), (False, 64), (False, 96)):
        w = wl.paper_wave(n0)
        H = oracle_mod.OracleHierarchy.from_workload(w)
        ns = int(round(T / w.dt_coarse))
        assert abs(ns * w.dt_coarse - T) < 1e-12
        for _ in range(ns):
            H.step(w.dt_coarse, sub)
        err[(sub, n0)] = [max(np.max(np.abs(H.read(l, 0, c) - wl.spherical_wave_exact(w, l, 0, c, T))) for c in (0, 1))
                          for l in range(3)]
    o_med = math.log(err[(True, 64)][2] / err[(True, 96)][2]) / math.log(1.5)
    o_high = math.log(err[(True, 64)][2] / err[(True, 128)][2]) / math.log(2.0)
    o_uni = math.log(err[(False, 64)][2] / err[(False, 96)][2]) / math.log(1.5)
    print("Fig. 1 orders (level 2): sub %.2f %.2f, uniform %.2f; errors %s" % (o_med, o_high, o_uni, err))
    assert 3.7 < o_med < 4.3 and 3.7 < o_high < 4.3 and 3.7 < o_uni < 4.3
    for n0 in (64, 96):  # subcycling and uniform stepping give the same error curve (Fig. 1)
        assert abs(err[(True, n0)][2] / err[(False, n0)][2] - 1.0) < 0.05


_FLOOR_SCRIPT = r"""
import sys, numpy as np
sys.path.insert(0, sys.argv[1])
import oracle
from paper_2503_09629_b200 import workloads as wl
w = wl.cfg5_spacings(32, 6)   # six levels with cfg 5's dx and dt on EVERY level: its 128 finest-level RHS evaluations
O = oracle.OracleHierarchy.from_workload(w)
O.step(w.dt_coarse, True)
assert oracle.lib().oc_real_bytes() == int(sys.argv[3])
np.savez(sys.argv[2], **{f"l{l}c{c}": O.read(l, 0, c, padded=True) for l in range(w.nlevels) for c in range(2)})
"""


def test_rounding_floor_of_the_oracle(tmp_path):
    """Reading S27: what a tolerance of 1e-11 max|u| can mean at cfg 5's depth, measured AT that
    depth. The same oracle source built three ways — as shipped (O64); with multiply-adds contracted (-mfma
    -ffp-contract=fast: every a*b+c rounds once instead of twice, nothing else changes); and with long double state and
    accumulators (-DORACLE_LONG_DOUBLE: 11 more mantissa bits, the exact-arithmetic value T at fp64 resolution) — takes
    one subcycled coarse step of six levels that have cfg 5's spacing and time step on every level (finest 2 / 8192, 128
    RHS evaluations there). Measured (32^3 boxes; 64^3 gives 7.9e-12 / 1.1e-11): u lies 7e-16 max|u| from T on every level; rho lies
    7.0e-12 max|u| from T on the finest level, and the two fp64 builds are 9.3e-12 max|u| apart: two correct fp64
    evaluations of the definition sit AT north_star's 1e-11 max|u| from each other in rho by rounding alone, so that
    bound cannot be applied to rho there. oracle/parity.py's analytic floor F (linear accumulation) is 3.6e-11 max|u|: the
    measured distance is 0.2 F. The GPU side of the argument — the CUDA result is as close to T as O64 is — is
    tests/test_gpu_truth.py."""
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "floor.py"
    script.write_text(_FLOOR_SCRIPT)
    variants = [("plain", "", 8), ("truth", "-DORACLE_LONG_DOUBLE", 16)]
    if "fma" in open("/proc/cpuinfo").read():
        variants.append(("fma", "-mfma -ffp-contract=fast", 8))
    out = {}
    for name, flags, nbytes in variants:
        env = dict(os.environ, ORACLE_SO=str(tmp_path / f"liboracle_{name}.so"), ORACLE_CXXFLAGS=flags)
        subprocess.run([sys.executable, str(script), root, str(tmp_path / f"{name}.npz"), str(nbytes)], check=True, env=env)
        out[name] = np.load(tmp_path / f"{name}.npz")
    a, t = out["plain"], out["truth"]
    nl = 6
    su = max(np.abs(t[f"l{l}c0"]).max() for l in range(nl))
    du = max(np.abs(a[f"l{l}c0"] - t[f"l{l}c0"]).max() for l in range(nl)) / su
    d_lvl = [np.abs(a[f"l{l}c1"] - t[f"l{l}c1"]).max() / su for l in range(nl)]
    from oracle.parity import rho_floor
    F = rho_floor(wl.cfg5_spacings(32, 6), su) / su
    print("rounding floor at cfg 5's depth: |O64 - T| u %.1e, rho per level %s, F %.1e" % (du, ["%.1e" % d for d in d_lvl], F))
    assert abs(F / 3.64e-11 - 1) < 0.01          # the analytic floor at this depth (oracle/parity.py): 128 eps 0.625 / dx
    assert du <= 5e-15                           # u: four orders inside 1e-11 max|u|
    assert 4e-12 <= d_lvl[5] <= 1.4e-11          # rho: fp64 is this far from the exact value (measured 7.0e-12) ...
    assert 0.1 * F <= d_lvl[5] <= 0.4 * F        # ... = 0.2 F: F bounds it with a factor 5 to spare, not 50
    assert d_lvl[5] > 20.0 * d_lvl[1]            # it is the depth that does it (eps 0.6 |u| / dx per evaluation)
    if "fma" in out:                             # two fp64 roundings of the same arithmetic: AT the literal bound
        b = out["fma"]
        dr = max(np.abs(a[f"l{l}c1"] - b[f"l{l}c1"]).max() for l in range(nl)) / su
        dtb = max(np.abs(b[f"l{l}c1"] - t[f"l{l}c1"]).max() for l in range(nl)) / su
        print("plain vs fma: %.1e; fma vs T: %.1e" % (dr, dtb))
        assert 5e-12 <= dr <= 2e-11 and dr <= d_lvl[5] + dtb and 4e-12 <= dtb <= 1.4e-11
