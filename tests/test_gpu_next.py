"""GPU parity of the NEXT-3 / NEXT-4 options against the CPU oracle, through the C ABI: RK3 / RK2 subcycling
(PAPER.md:359, S28), the radiative outer boundary, 8th-order differences with fifth- and ninth-order
dissipation (eq 36), the 9-/10-point interpolation (S30) and vertex-centred grids (S31), alone and
combined, in both modes, ghosts included. Tolerance: oracle/parity.py. Plus closed forms with no oracle involved."""
import math

import numpy as np
import pytest

import oracle
import paper_2503_09629_b200 as sc
from oracle.parity import compare_state
from paper_2503_09629_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _run_pair(w, sub, steps=None):
    G, O = sc.Hierarchy.from_workload(w), oracle.OracleHierarchy.from_workload(w)
    n = w.coarse_steps if steps is None else steps
    for _ in range(n):
        G.sc_step(w.dt_coarse, sub)
        O.step(w.dt_coarse, sub)
    rel = compare_state(G, O, w, what=f"{w.name} sub={sub}")  # nsteps = 1: the strictest floors (shallow hierarchies: F is nothing)
    G.close()
    return rel


def _three_levels(**opt):
    """Non-cubic three-level hierarchy with margins wide enough for every interpolation variant (>= 7 parent cells)."""
    boxes = [wl.Box(0, (0, 0, 0), (48, 40, 44)), wl.Box(1, (20, 16, 18), (56, 48, 52)), wl.Box(2, (56, 48, 52), (24, 20, 22)),
             wl.Box(2, (96, 52, 56), (20, 24, 18))]
    w = wl.Workload("3 levels " + " ".join(f"{k}={v}" for k, v in opt.items()), boxes, (48, 40, 44),
                    xlo=(-1.0, -0.8, -0.9), xhi=(1.0, 0.8, 0.9), coarse_steps=2, init=wl.multi_gaussian_init(3))
    for k, v in opt.items():
        setattr(w, k, v)
    return w


@pytest.mark.parametrize("integ", [3, 2])
@pytest.mark.parametrize("sub", [True, False])
def test_rk3_rk2_parity(integ, sub):
    """cfg 1 (8 steps), the ragged coupled multi-box hierarchy and a 4-level hierarchy with the lower-order integrators,
    with and without dissipation."""
    for w in (wl.cfg1(), wl.ragged_small(), wl.cfg3(32, 4)):
        for sigma in (0.0, 0.2):
            w.integrator, w.ko_sigma = integ, sigma
            w.coarse_steps = min(w.coarse_steps, 3)
            _run_pair(w, sub)


@pytest.mark.parametrize("integ", [4, 3, 2])
@pytest.mark.parametrize("sub", [True, False])
def test_radiative_boundary_parity(integ, sub):
    """Radiative outer boundary on a 3-level hierarchy and on one level, every integrator, with dissipation on and off."""
    for sigma in (0.0, 0.15):
        _run_pair(_three_levels(outer_bc=1, integrator=integ, ko_sigma=sigma), sub)
    n = 32
    one = wl.Workload("one level radiative", [wl.Box(0, (0, 0, 0), (n, n, n))], (n, n, n), xlo=(-2.0,) * 3, xhi=(2.0,) * 3,
                      outer_bc=1, integrator=integ, coarse_steps=6,
                      init=lambda w, l, ib, c: wl.spherical_wave_exact(w, l, ib, c, 0.0, 0.35))
    _run_pair(one, sub)


@pytest.mark.parametrize("sub", [True, False])
def test_fd8_with_dissipation_parity(sub):
    """8th-order differences with ninth-order dissipation at g = 5 (eq 36 with r = 8) and with fifth-order dissipation at
    g = 4 (the pair every spacetime run of the paper uses), coupled fields included."""
    _run_pair(_three_levels(fd_order=8, ghost=5, ko_sigma=0.2, ko_order=9), sub)
    _run_pair(_three_levels(fd_order=8, ghost=4, ko_sigma=0.2, ko_order=5), sub)
    w = wl.ragged_small()
    w.fd_order, w.ghost, w.ko_sigma, w.ko_order = 8, 4, 0.25, 5
    _run_pair(w, sub)
    w = wl.cfg1()
    w.fd_order, w.ghost, w.ko_sigma = 8, 5, 0.25
    _run_pair(w, sub, steps=3)


@pytest.mark.parametrize("interp,vertex,ghost,fd", [(1, 0, 4, 8), (1, 0, 5, 8), (0, 1, 3, 4), (1, 1, 4, 8), (0, 0, 5, 4)])
@pytest.mark.parametrize("sub", [True, False])
def test_interpolation_variants_parity(interp, vertex, ghost, fd, sub):
    """9-point prolongation / 10-point restriction, vertex-centred grids with injection, and the quartic operator at
    g = 5 — on the two-launch path (no dissipation) and on the general path (with it)."""
    _run_pair(_three_levels(interp=interp, vertex=vertex, ghost=ghost, fd_order=fd), sub)
    if ghost >= 3:
        _run_pair(_three_levels(interp=interp, vertex=vertex, ghost=ghost, fd_order=fd, ko_sigma=0.2, ko_order=5), sub)


def test_everything_together_parity():
    """RK3 + radiative boundary + 8th-order differences + ninth-order dissipation + 9-/10-point interpolation, g = 5."""
    _run_pair(_three_levels(integrator=3, outer_bc=1, fd_order=8, ghost=5, ko_sigma=0.2, interp=1), True)
    _run_pair(_three_levels(integrator=2, outer_bc=1, fd_order=8, ghost=5, ko_sigma=0.2, vertex=1), True)


def test_vertex_ghost_index_map_bit_exact():
    w = _three_levels(vertex=1)
    G, O = sc.Hierarchy.from_workload(w), oracle.OracleHierarchy.from_workload(w)
    for ib in (0, 1):
        assert np.array_equal(G.sc_debug_ghost_map(2, ib), O.ghost_map(2, ib))
    G.close()


@pytest.mark.parametrize("integ", [3, 2])
def test_rk_closed_forms_without_the_oracle(integ):
    """The CUDA path against closed forms: (i) one periodic level on a Fourier mode: n steps apply R(dt M)^n with the
    integrator's stability polynomial; (ii) the exact quadratic solution through 3 subcycled levels."""
    n = 16
    w = wl.Workload("t", [wl.Box(0, (0, 0, 0), (n, n, n))], (n, n, n), integrator=integ, init=lambda *a: np.zeros((n, n, n)))
    G = sc.Hierarchy.from_workload(w)
    x, y, z = w.centres(0, 0)
    kv = math.pi * np.array([1, 2, -1])
    ph = kv[2] * z[:, None, None] + kv[1] * y[None, :, None] + kv[0] * x[None, None, :]
    s, c = np.sin(ph), np.cos(ph)
    G.sc_set_state(0, 0, 0, 0.7 * s - 0.2 * c)
    G.sc_set_state(0, 0, 1, 1.1 * s + 0.4 * c)
    h = w.dx(0)
    kappa2 = sum((30 - 32 * math.cos(k * h) + 2 * math.cos(2 * k * h)) / (12 * h * h) for k in kv)
    dt, nsteps = 0.25 * h, 30
    Z = dt * np.array([[0.0, 1.0], [-kappa2, 0.0]])
    R1, P = np.eye(2), np.eye(2)
    for m in range(1, integ + 1):
        P = P @ Z / m
        R1 = R1 + P
    R = np.linalg.matrix_power(R1, nsteps)
    for _ in range(nsteps):
        G.sc_step(dt, True)
    a, b = R @ np.array([0.7, 1.1])
    cc, d = R @ np.array([-0.2, 0.4])
    assert np.max(np.abs(G.sc_read_level(0, 0, 0) - (a * s + cc * c))) < 5e-13
    assert np.max(np.abs(G.sc_read_level(0, 0, 1) - (b * s + d * c))) < 5e-12
    G.close()
    n = 48
    w = wl.Workload("quadratic", wl.nested_cubes(3, n), (n, n, n), init=wl.quadratic_init, integrator=integ)
    G = sc.Hierarchy.from_workload(w)
    G.sc_step(w.dt_coarse, True)
    for l in (1, 2):
        for comp in (0, 1):
            got = G.sc_debug_read_padded(l, 0, comp)
            assert np.max(np.abs(got - wl.quadratic_exact(w, l, 0, comp, w.dt_coarse, pad=w.ghost))) < 5e-12, (l, comp)
    G.close()


def test_radiative_pulse_leaves_the_box_without_the_oracle():
    """The paper's spherical wave on [-2,2]^3 to t = 3.2 with the radiative boundary on the CUDA path alone: the error
    against the exact outgoing solution is a few per cent of the pulse at 32^3 and falls faster than second order."""
    errs = []
    for n in (32, 64):
        w = wl.Workload("pulse", [wl.Box(0, (0, 0, 0), (n, n, n))], (n, n, n), xlo=(-2.0,) * 3, xhi=(2.0,) * 3, outer_bc=1,
                        init=lambda w_, l, ib, c: wl.spherical_wave_exact(w_, l, ib, c, 0.0, 0.35))
        G = sc.Hierarchy.from_workload(w)
        steps = int(round(3.2 / w.dt_coarse))
        for _ in range(steps):
            G.sc_step(w.dt_coarse, True)
        errs.append(float(np.max(np.abs(G.sc_read_level(0, 0, 0) - wl.spherical_wave_exact(w, 0, 0, 0, steps * w.dt_coarse, 0.35)))))
        G.close()
    assert errs[0] < 0.05 and errs[1] < errs[0] / 3.0, errs


@pytest.mark.parametrize("g,interp,vertex,fd", [(5, 0, 0, 4), (4, 1, 0, 8), (5, 1, 0, 8), (3, 0, 1, 4), (5, 1, 1, 8), (2, 0, 1, 4)])
def test_general_ghost_and_restriction_geometry_sweep(g, interp, vertex, fd):
    """The general separable ghost fill / restriction (ghost_gen.cu) on child boxes of every offset class (lo mod 4 per
    axis), sizes that are no multiple of its 16 x 16 tiles or its 8 x 8 x 4 restriction tiles, the smallest box (n = 8) and
    a child that reaches the nesting margin of each variant: one subcycled + one uniform step, every ghost and interior
    value against the oracle, index map bit-exact."""
    B = wl.Box
    margin = (g + 1) // 2 + (2, 4, 3, 5)[interp + 2 * vertex]
    cases = [
        ((40, 32, 36), (2 * margin, 2 * margin, 2 * margin), (80 - 4 * margin, 64 - 4 * margin, 72 - 4 * margin)),  # child up to the margin on every side
        ((64, 64, 64), (22, 20, 26), (44, 28, 18)),
        ((64, 64, 64), (20, 22, 24), (30, 46, 34)),
        ((48, 40, 36), (30, 26, 22), (8, 8, 8)),
        ((36, 36, 36), (18, 22, 20), (20, 14, 34)),
    ]
    for dom, lo, n in cases:
        w = wl.Workload(f"sweep {dom} {lo} {n} g={g} interp={interp} vertex={vertex}", [B(0, (0, 0, 0), dom), B(1, lo, n)], dom,
                        ghost=g, interp=interp, vertex=vertex, fd_order=fd, init=wl.multi_gaussian_init(3))
        G, O = sc.Hierarchy.from_workload(w), oracle.OracleHierarchy.from_workload(w)
        for sub in (True, False):
            G.sc_step(w.dt_coarse, sub)
            O.step(w.dt_coarse, sub)
            compare_state(G, O, w, what=w.name + f" sub={sub}")
        assert np.array_equal(G.sc_debug_ghost_map(1, 0), O.ghost_map(1, 0))
        G.close()
