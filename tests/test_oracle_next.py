"""Pins for the oracle's NEXT-3 / NEXT-4 options: RK3 / RK2 subcycling (reading S28),
the radiative outer boundary, ninth-order Kreiss-Oliger dissipation with 8th-order differences
(eq 36 with r = 8), interpolation operators that follow the 8th-order stencil (S30) and vertex-centred
grids with injection (S31). CPU only.

What fixes the expected values: the order conditions of Runge-Kutta continuous extensions, the stability polynomials
1 + z + z^2/2 (+ z^3/6), a scalar ODE integrated by hand in this file, the exact polynomial and spherical-wave
solutions of the wave equation, the closed-form symbol -(2 - 2 cos kh)^5 of delta^10, polynomial exactness, and
floating-point geometry for the index maps."""
import math

import numpy as np
import pytest

from paper_2503_09629_b200 import workloads as wl

TABLEAU = {  # (c, b, A) of the integrators of reading S28, typed here from the textbook tableaux
    4: ([0, .5, .5, 1], [1 / 6, 1 / 3, 1 / 3, 1 / 6], [[0] * 4, [.5, 0, 0, 0], [0, .5, 0, 0], [0, 0, 1, 0]]),
    3: ([0, .5, 1], [1 / 6, 2 / 3, 1 / 6], [[0] * 3, [.5, 0, 0], [-1, 2, 0]]),
    2: ([0, .5], [0, 1], [[0] * 2, [.5, 0]]),
}


# ----------------------------------------------------------------------------------------------
# RK3 / RK2 dense output and ghost stage vectors
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("integ", [3, 2])
def test_rk_dense_output_order_conditions(oracle_mod, integ):
    """b_i(0) = 0, b_i(1) = the method's weights, and the order conditions of a continuous extension (Hairer-Norsett-
    Wanner II.6): sum b_i = theta, sum b_i c_i = theta^2/2 for both; for RK3 — whose dense output uses the extra
    slope k4 = f(y_{n+1}), i.e. the row (1/6, 2/3, 1/6) with c_4 = 1 — also sum b_i c_i^2 = theta^3/3 and
    sum_i b_i sum_j a_ij c_j = theta^3/6 (third order). Derivatives against central differences of b itself."""
    c, bw, A = TABLEAU[integ]
    S = integ
    if integ == 3:  # the extended tableau of the dense output
        c, bw, A, S = c + [1], bw + [0], [r + [0] for r in A] + [bw + [0]], 4
    for th in (0.0, 0.25, 0.5, 0.7, 1.0):
        b = [oracle_mod.b_rk(integ, i + 1, 0, th) for i in range(S)]
        assert abs(sum(b) - th) < 1e-15
        assert abs(sum(bi * ci for bi, ci in zip(b, c)) - th * th / 2) < 1e-15
        if integ == 3:
            assert abs(sum(bi * ci * ci for bi, ci in zip(b, c)) - th ** 3 / 3) < 1e-15
            assert abs(sum(b[i] * sum(A[i][j] * c[j] for j in range(S)) for i in range(S)) - th ** 3 / 6) < 1e-15
        for i in range(S):
            for m in (1, 2):
                e = 1e-4
                fd = (oracle_mod.b_rk(integ, i + 1, m - 1, th + e) - oracle_mod.b_rk(integ, i + 1, m - 1, th - e)) / (2 * e)
                assert abs(fd - oracle_mod.b_rk(integ, i + 1, m, th)) < 1e-7, (i, m, th)
    assert all(abs(oracle_mod.b_rk(integ, i + 1, 0, 0.0)) == 0.0 for i in range(S))
    assert np.allclose([oracle_mod.b_rk(integ, i + 1, 0, 1.0) for i in range(S)], bw, atol=1e-15)


def _f(y):
    return -y * y + math.sin(y)


def _rk_stages(integ, y, h):
    """Stage vectors Y_1..Y_S, slopes and the update of one step of size h from y (scalar ODE y' = _f(y))."""
    _, b, A = TABLEAU[integ]
    Y, k = [], []
    for s in range(integ):
        Ys = y + h * sum(A[s][j] * k[j] for j in range(s))
        Y.append(Ys)
        k.append(_f(Ys))
    return Y, k, y + h * sum(bi * ki for bi, ki in zip(b, k))


@pytest.mark.parametrize("integ", [3, 2])
def test_rk_theta_one_reproduces_update_and_ghost_stage_order(oracle_mod, integ):
    """(i) The dense output at theta = 1 is the method's own update. (ii) Scalar ODE y' = -y^2 + sin y: the ghost stage
    vectors built from the PARENT's slopes (step hp) for a child step h = hp/2 starting at theta = 0 and 1/2 against the
    stage vectors the child's own integrator computes from the same start value: the difference must shrink like
    h^4 (RK3: stages 2, 3, as eqs 15-18 do for RK4) / h^2 (RK2: stage 2)."""
    y0 = 0.8
    errs = {}
    for hp in (0.2, 0.1, 0.05):
        _, k, ynew = _rk_stages(integ, y0, hp)
        if integ == 3:
            k = k + [_f(ynew)]  # the dense output's extra slope
        assert abs(oracle_mod.dense_stage_rk(integ, 5, 1.0, hp, y0, k) - ynew) < 1e-15
        assert oracle_mod.dense_stage_rk(integ, 1, 0.0, hp, y0, k) == y0
        for th in (0.0, 0.5):
            ystart = oracle_mod.dense_stage_rk(integ, 1, th, hp, y0, k)
            Y, _, _ = _rk_stages(integ, ystart, hp / 2)
            for s in range(2, integ + 1):
                errs.setdefault((th, s), []).append(abs(oracle_mod.dense_stage_rk(integ, s, th, hp, y0, k) - Y[s - 1]))
    need = 3.6 if integ == 3 else 1.8
    assert max(errs[(0.0, 2)]) < 1e-15  # theta = 0: y' = k_1 exactly, the ghost Y_2 IS the child's Y_2
    for key, e in errs.items():
        if key == (0.0, 2):
            continue
        assert e[0] > 0 and math.log2(e[0] / e[1]) > need and math.log2(e[1] / e[2]) > need, (key, e)


def _stab(integ, Z):
    R, P = np.eye(2), np.eye(2)
    for m in range(1, integ + 1):
        P = P @ Z / m
        R = R + P
    return R


@pytest.mark.parametrize("integ", [3, 2])
def test_rk_single_level_closed_form_amplification(oracle_mod, integ):
    """One periodic level on a Fourier mode: n steps apply R(dt M)^n with the integrator's stability polynomial
    R = 1 + z + z^2/2 (+ z^3/6) — pins the tableau (a wrong stage coefficient or weight changes R)."""
    n = 16
    w = wl.Workload("t", [wl.Box(0, (0, 0, 0), (n, n, n))], (n, n, n), integrator=integ, init=lambda *a: np.zeros((n, n, n)))
    H = oracle_mod.OracleHierarchy.from_workload(w)
    x, y, z = w.centres(0, 0)
    kv = math.pi * np.array([1, 2, -1])
    ph = kv[2] * z[:, None, None] + kv[1] * y[None, :, None] + kv[0] * x[None, None, :]
    s, c = np.sin(ph), np.cos(ph)
    H.set_state(0, 0, 0, 0.7 * s - 0.2 * c)
    H.set_state(0, 0, 1, 1.1 * s + 0.4 * c)
    h = w.dx(0)
    kappa2 = sum((30 - 32 * math.cos(k * h) + 2 * math.cos(2 * k * h)) / (12 * h * h) for k in kv)
    dt, nsteps = 0.25 * h, 30
    R = np.linalg.matrix_power(_stab(integ, dt * np.array([[0.0, 1.0], [-kappa2, 0.0]])), nsteps)
    for _ in range(nsteps):
        H.step(dt, True)
    a, b = R @ np.array([0.7, 1.1])
    cc, d = R @ np.array([-0.2, 0.4])
    assert np.max(np.abs(H.read_level(0, 0, 0) - (a * s + cc * c))) < 2e-13
    assert np.max(np.abs(H.read_level(0, 0, 1) - (b * s + d * c))) < 2e-12
    R4 = np.linalg.matrix_power(_stab(4, dt * np.array([[0.0, 1.0], [-kappa2, 0.0]])), nsteps)
    assert abs((R4 @ np.array([0.7, 1.1]))[0] - a) > 1e-7  # RK4 would give a different answer


@pytest.mark.parametrize("integ", [3, 2])
@pytest.mark.parametrize("sub", [True, False])
def test_rk_composite_scheme_exact_for_quadratic_solution(oracle_mod, integ, sub):
    """u = r^2 + 3 t^2, rho = 6 t through one coarse step of a 3-level hierarchy: RK3 and RK2 integrate a solution
    quadratic in t exactly, their dense outputs and the ghost stage formulas of S28 reproduce it exactly for a linear
    autonomous system (k2 = y' + h/2 y'' and f(y + d) = f(y) + f_y d hold exactly), so every level must return the
    polynomial to rounding — theta = 0 and 1/2 fills, stage vectors in the ghosts, restrictions, both modes."""
    n = 48
    w = wl.Workload("quadratic", wl.nested_cubes(3, n), (n, n, n), init=wl.quadratic_init, integrator=integ)
    H = oracle_mod.OracleHierarchy.from_workload(w)
    H.step(w.dt_coarse, sub)
    t = w.dt_coarse
    for l in (1, 2):
        for c in (0, 1):
            got = H.read(l, 0, c, padded=True)
            want = wl.quadratic_exact(w, l, 0, c, t, pad=w.ghost)
            assert np.max(np.abs(got - want)) < 2e-12, (integ, sub, l, c, float(np.max(np.abs(got - want))))
    m = slice(10, n - 10)
    for c in (0, 1):
        assert np.max(np.abs(H.read(0, 0, c)[m, m, m] - wl.quadratic_exact(w, 0, 0, c, t)[m, m, m])) < 2e-12


def _plane_errors(oracle_mod, n, sub, t_end=0.5, **opt):
    w = wl.cfg2(n)
    if opt.get("vertex"):  # the 6-point midpoint stencil reaches one parent point further: margin 5 instead of 4
        w.boxes[1] = wl.Box(1, (n // 2 + 2,) * 3, (n - 4,) * 3)
    for k, v in opt.items():
        setattr(w, k, v)
    H = oracle_mod.OracleHierarchy.from_workload(w)
    steps = int(round(t_end / w.dt_coarse))
    for _ in range(steps):
        H.step(w.dt_coarse, sub)
    t = steps * w.dt_coarse
    return [np.max(np.abs(H.read_level(l, 0, 0) - wl.plane_wave_exact(w, l, 0, 0, t))) for l in (0, 1)]


@pytest.mark.slow
@pytest.mark.parametrize("integ,order", [(3, 3.0), (2, 2.0)])
def test_rk_convergence_ladder(oracle_mod, integ, order):
    """cfg-2 ladder (two levels, exact plane wave) with the lower-order integrators: the subcycled scheme converges at
    the integrator's order (measured: RK3 3.33 / 3.18 for 16 -> 32 -> 64, RK2 1.92 / 1.97), and the subcycled error stays
    within a small factor of the uniform one (which takes the fine step everywhere)."""
    e16 = _plane_errors(oracle_mod, 16, True, integrator=integ)
    e32 = _plane_errors(oracle_mod, 32, True, integrator=integ)
    u32 = _plane_errors(oracle_mod, 32, False, integrator=integ)
    for l in (0, 1):
        o = math.log2(e16[l] / e32[l])
        assert order - 0.35 < o < order + 0.6, (integ, l, e16, e32, o)
        assert u32[l] < e32[l] < 6.0 * u32[l], (e32, u32)  # coarser steps on level 0: larger, same magnitude


# ----------------------------------------------------------------------------------------------
# radiative outer boundary
# ----------------------------------------------------------------------------------------------
def test_radiative_rhs_exact_for_quadratics(oracle_mod):
    """k_1 of a step = f(y_n). With a radiative outer boundary the cells within g of a face obey
    d_t y = -(x.grad y + y)/r (S29), and the second-order centred / one-sided differences are exact for quadratics:
    on y = p(x,y,z) of degree 2 the slope must equal -(x.grad p + p)/r to rounding in the whole boundary zone, for u AND
    rho, while the cells further in keep the interior formulas (k_u = rho, k_rho = Lap u)."""
    n, g = (20, 16, 24), 3
    w = wl.Workload("rad", [wl.Box(0, (0, 0, 0), n)], n, xlo=(-1.0, -0.8, -1.2), xhi=(1.0, 0.8, 1.2), outer_bc=1,
                    init=lambda *a: np.zeros((n[2], n[1], n[0])))
    H = oracle_mod.OracleHierarchy.from_workload(w)
    x, y, z = w.centres(0, 0)
    X, Y, Z = x[None, None, :], y[None, :, None], z[:, None, None]

    def quad(c):
        p = c[0] + c[1] * X + c[2] * Y + c[3] * Z + c[4] * X * X + c[5] * Y * Y + c[6] * Z * Z + c[7] * X * Y + c[8] * Y * Z + c[9] * X * Z
        gx = c[1] + 2 * c[4] * X + c[7] * Y + c[9] * Z
        gy = c[2] + 2 * c[5] * Y + c[7] * X + c[8] * Z
        gz = c[3] + 2 * c[6] * Z + c[8] * Y + c[9] * X
        return p + 0 * (X + Y + Z), gx + 0 * (X + Y + Z), gy + 0 * (X + Y + Z), gz + 0 * (X + Y + Z), 2 * (c[4] + c[5] + c[6])
    cu = [.3, -1, .5, 2, 1, -.7, .2, .9, -.4, .6]
    cr = [-.8, .4, 1.5, -.3, .5, .25, -1.1, .3, .7, -.2]
    pu, *gu, lapu = quad(cu)
    pr, *gr, _ = quad(cr)
    H.set_state(0, 0, 0, pu)
    H.set_state(0, 0, 1, pr)
    H.step(1e-9, True)
    k1u, k1r = H.read(0, 0, 0, slot=2), H.read(0, 0, 1, slot=2)
    r = np.sqrt(X * X + Y * Y + Z * Z)
    zone = np.zeros(pu.shape, bool)
    for ax, nn in ((2, n[0]), (1, n[1]), (0, n[2])):
        idx = np.arange(nn)
        m = (idx < g) | (idx >= nn - g)
        sh = [1, 1, 1]
        sh[ax] = nn
        zone |= m.reshape(sh)
    want_u = -(X * gu[0] + Y * gu[1] + Z * gu[2] + pu) / r
    want_r = -(X * gr[0] + Y * gr[1] + Z * gr[2] + pr) / r
    assert zone.sum() > 0 and (~zone).sum() > 0
    assert np.max(np.abs(k1u - want_u)[zone]) < 1e-11
    assert np.max(np.abs(k1r - want_r)[zone]) < 1e-11
    assert np.max(np.abs(k1u - pr)[~zone]) < 1e-13          # interior: k_u = rho
    assert np.max(np.abs(k1r - lapu)[~zone]) < 1e-9         # interior: k_rho = Lap u (exact for quadratics)
    assert np.max(np.abs(want_u - pr)[zone]) > 0.1           # the two formulas differ: the zone mask is being tested


def _outgoing_error(oracle_mod, n, outer_bc, t_end, sigma=0.35):
    w = wl.Workload("pulse", [wl.Box(0, (0, 0, 0), (n, n, n))], (n, n, n), xlo=(-2.0,) * 3, xhi=(2.0,) * 3,
                    outer_bc=outer_bc, init=lambda w, l, ib, c: wl.spherical_wave_exact(w, l, ib, c, 0.0, sigma))
    H = oracle_mod.OracleHierarchy.from_workload(w)
    steps = int(round(t_end / w.dt_coarse))
    for _ in range(steps):
        H.step(w.dt_coarse, True)
    return float(np.max(np.abs(H.read_level(0, 0, 0) - wl.spherical_wave_exact(w, 0, 0, 0, steps * w.dt_coarse, sigma))))


@pytest.mark.slow
def test_radiative_boundary_lets_the_pulse_leave(oracle_mod):
    """The paper's spherical wave (eqs 41-42, wider pulse) on [-2,2]^3, run to t = 3.2, when the exact solution has
    left the box. An outgoing wave f(t-r)/r satisfies d_t y + (x/r).grad y + y/r = 0 exactly, so with the radiative
    boundary the numerical solution follows the exact one up to the O(h^2) boundary differences: the error is a small
    fraction of the pulse amplitude (peak |u| ~ 1.7 at t = 0.4) and falls at second order; with the periodic boundary
    the pulse re-enters and the error is of the order of the solution itself."""
    e32 = _outgoing_error(oracle_mod, 32, 1, 3.2)
    e64 = _outgoing_error(oracle_mod, 64, 1, 3.2)
    p32 = _outgoing_error(oracle_mod, 32, 0, 3.2)
    assert e32 < 0.05 and e64 < e32 / 3.0, (e32, e64)   # measured 3.4e-2 / 2.8e-3
    assert p32 > 10 * e32, (p32, e32)


# ----------------------------------------------------------------------------------------------
# 8th-order differences with ninth-order dissipation (g = 5)
# ----------------------------------------------------------------------------------------------
def test_fd8_with_ninth_order_dissipation_closed_form(oracle_mod):
    """Eq (36) with r = 8: on a Fourier mode Q is the number q = -sigma/1024 sum_axis (2 - 2 cos kh)^5 / h (the symbol of
    delta^10 = (D+D-)^5 h^10 is -(2 sin kh/2)^10; q = -sigma/h per axis at the Nyquist mode), acting on u and rho:
    M = [[q, 1], [-kappa8^2, q]] with the 9-point symbol of the second difference."""
    n, sigma = 16, 0.25
    zero = lambda *a: np.zeros((n, n, n))  # noqa: E731
    w = wl.Workload("t", [wl.Box(0, (0, 0, 0), (n, n, n))], (n, n, n), ghost=5, ko_sigma=sigma, fd_order=8, ko_order=9, init=zero)
    H = oracle_mod.OracleHierarchy.from_workload(w)
    x, y, z = w.centres(0, 0)
    kv = math.pi * np.array([3, -2, 5])
    ph = kv[2] * z[:, None, None] + kv[1] * y[None, :, None] + kv[0] * x[None, None, :]
    s, c = np.sin(ph), np.cos(ph)
    H.set_state(0, 0, 0, 0.7 * s - 0.2 * c)
    H.set_state(0, 0, 1, 1.1 * s + 0.4 * c)
    h = w.dx(0)
    c8 = [-205 / 72, 8 / 5, -1 / 5, 8 / 315, -1 / 560]
    kappa2 = -sum((c8[0] + 2 * sum(c8[m] * math.cos(m * k * h) for m in range(1, 5))) / (h * h) for k in kv)
    q = -sigma / 1024.0 * sum((2 - 2 * math.cos(k * h)) ** 5 / h for k in kv)
    dt, nsteps = 0.25 * h, 20
    Z = dt * np.array([[q, 1.0], [-kappa2, q]])
    R = np.linalg.matrix_power(_stab(4, Z), nsteps)
    for _ in range(nsteps):
        H.step(dt, True)
    a, b = R @ np.array([0.7, 1.1])
    cc, d = R @ np.array([-0.2, 0.4])
    assert np.max(np.abs(H.read_level(0, 0, 0) - (a * s + cc * c))) < 2e-13
    assert np.max(np.abs(H.read_level(0, 0, 1) - (b * s + d * c))) < 2e-12
    # fifth-order dissipation on the same stencil (the paper's production pair) is a different number
    w5 = wl.Workload("t", w.boxes, w.domain_cells, ghost=5, ko_sigma=sigma, fd_order=8, ko_order=5, init=zero)
    H5 = oracle_mod.OracleHierarchy.from_workload(w5)
    H5.set_state(0, 0, 0, 0.7 * s - 0.2 * c)
    H5.set_state(0, 0, 1, 1.1 * s + 0.4 * c)
    for _ in range(nsteps):
        H5.step(dt, True)
    q5 = sigma / 64.0 * sum((2 * math.cos(3 * k * h) - 12 * math.cos(2 * k * h) + 30 * math.cos(k * h) - 20) / h for k in kv)
    R5 = np.linalg.matrix_power(_stab(4, dt * np.array([[q5, 1.0], [-kappa2, q5]])), nsteps)
    a5, _ = R5 @ np.array([0.7, 1.1])
    c5, _ = R5 @ np.array([-0.2, 0.4])
    assert np.max(np.abs(H5.read_level(0, 0, 0) - (a5 * s + c5 * c))) < 2e-13
    assert abs(a5 - a) > 1e-4


@pytest.mark.parametrize("sub", [True, False])
def test_fd8_ko9_composite_exact_for_quadratic_solution(oracle_mod, sub):
    """delta^10 annihilates polynomials of degree <= 9 and the 9-point second difference is exact to degree 9: the exact
    quadratic solution survives the composite 3-level step with g = 5, all five ghost layers filled at every stage."""
    # level 0's periodic seam spoils 5 cells per RHS evaluation, 20 per step: the child's footprint (parent cells 21..42)
    # stays clear of it
    boxes = [wl.Box(0, (0, 0, 0), (64, 64, 64)), wl.Box(1, (52, 52, 52), (24, 24, 24)), wl.Box(2, (116, 116, 116), (24, 24, 24))]
    w = wl.Workload("quadratic fd8+KO9", boxes, (64, 64, 64), ghost=5, init=wl.quadratic_init, ko_sigma=0.2,
                    fd_order=8, ko_order=9)
    H = oracle_mod.OracleHierarchy.from_workload(w)
    H.step(w.dt_coarse, sub)
    t = w.dt_coarse
    for l in (1, 2):
        for c in (0, 1):
            got = H.read(l, 0, c, padded=True)
            assert np.max(np.abs(got - wl.quadratic_exact(w, l, 0, c, t, pad=w.ghost))) < 5e-12, (sub, l, c)


# ----------------------------------------------------------------------------------------------
# interpolation operators that follow the stencil; vertex-centred grids
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("interp,vertex,deg_p,deg_r", [(1, 0, 8, 9), (0, 1, 5, None), (1, 1, 9, None)])
def test_interp_variants_polynomial_exactness(oracle_mod, interp, vertex, deg_p, deg_r):
    """Weights: sum to 1; the prolongation is exact for monomials up to degree deg_p and NOT for deg_p + 1, the
    restriction up to deg_r and not deg_r + 1 (injection: exact for anything), evaluated at the geometric position of
    the fine / parent point. Vertex grids: the 6-point midpoint operator is the textbook (3,-25,150,150,-25,3)/256."""
    omin, w, rmin, r = oracle_mod.interp_weights(interp, vertex)
    np_ = w.shape[1]
    nodes = np.arange(omin, omin + np_, dtype=float)
    pos = (0.0, 0.5) if vertex else (-0.25, 0.25)
    for par in (0, 1):
        assert abs(w[par].sum() - 1) < 1e-13
        for d in range(deg_p + 2):
            err = abs(w[par] @ nodes ** d - pos[par] ** d)
            if vertex and par == 0:
                assert err < 1e-13
            elif d <= deg_p:
                assert err < 1e-9 * max(1.0, abs(nodes).max() ** d), (par, d, err)
            else:
                assert err > 1e-4, (par, d, err)
    if vertex:
        assert rmin == 0 and list(r) == [1.0]
        assert list(w[0]) == [1.0 if o == 0 else 0.0 for o in range(omin, omin + np_)]
        if interp == 0:
            assert np.allclose(w[1] * 256, [3, -25, 150, 150, -25, 3], atol=1e-12)
    else:
        fn = np.arange(rmin, rmin + len(r), dtype=float) - 0.5  # fine centres in fine spacings from the parent centre
        assert abs(r.sum() - 1) < 1e-13
        for d in range(deg_r + 2):
            err = abs(r @ fn ** d - (1.0 if d == 0 else 0.0))
            assert (err < 1e-9 * abs(fn).max() ** d) if d <= deg_r else (err > 1e-2), (d, err)
        assert np.allclose(w[0], w[1][::-1])


@pytest.mark.parametrize("interp,vertex,ghost,fd", [(1, 0, 4, 8), (0, 1, 3, 4), (1, 1, 4, 8)])
@pytest.mark.parametrize("sub", [True, False])
def test_interp_variants_whole_hierarchy_on_polynomials(oracle_mod, interp, vertex, ghost, fd, sub):
    """Index maps + operators through the hierarchy (as test_prolongation_and_restriction_exact_for_quartics): for u = a
    tensor quartic and a vanishing step the child's ghosts must hold the polynomial at the ghost positions and the
    covered parent cells must hold it at theirs — for the 9-/10-point operators and for vertex-centred grids, where
    'position' is the grid point xlo + i dx (S31) and the restriction is injection."""
    boxes = [wl.Box(0, (0, 0, 0), (48, 40, 44)), wl.Box(1, (20, 16, 18), (44, 40, 42)), wl.Box(2, (56, 48, 52), (24, 20, 22))]
    w = wl.Workload("t", boxes, (48, 40, 44), ghost=ghost, interp=interp, vertex=vertex, fd_order=fd,
                    xlo=(-1.0, -0.8, -0.9), xhi=(1.0, 0.8, 0.9))
    H = oracle_mod.OracleHierarchy.from_workload(
        wl.Workload("t", boxes, w.domain_cells, ghost=ghost, interp=interp, vertex=vertex, fd_order=fd, xlo=w.xlo, xhi=w.xhi,
                    init=lambda w_, l, ib, c: np.zeros(tuple(reversed(w_.box(l, ib).n)))))
    cx, cy, cz = [1, -2, .5, 3, -1], [.3, 1, -1, .5, 2], [2, .1, -.7, 1, 1]

    def poly(x, y, z, a, b, c):
        f = lambda v, co: sum(q * v ** m for m, q in enumerate(co))  # noqa: E731
        return f(z, c)[:, None, None] * f(y, b)[None, :, None] * f(x, a)[None, None, :]
    for l in range(3):
        x, y, z = w.centres(l, 0)
        H.set_state(l, 0, 0, poly(x, y, z, cx, cy, cz))
        H.set_state(l, 0, 1, poly(x, y, z, cz, cx, cy))
    H.step(1e-10, sub)
    for l in (1, 2):
        x, y, z = w.centres(l, 0, pad=ghost)
        for comp, cc in ((0, (cx, cy, cz)), (1, (cz, cx, cy))):
            assert np.max(np.abs(H.read(l, 0, comp, padded=True) - poly(x, y, z, *cc))) < 1e-8, (l, comp)
    b1 = w.box(1, 0)
    x, y, z = w.centres(0, 0)
    sl = tuple(slice(b1.lo[a] // 2, (b1.lo[a] + b1.n[a]) // 2) for a in (2, 1, 0))
    assert np.max(np.abs(H.read(0, 0, 0)[sl] - poly(x, y, z, cx, cy, cz)[sl])) < 1e-8


def test_vertex_ghost_index_map_brute_force_geometry(oracle_mod):
    """Vertex-centred grids (S31): fine point I sits at I dx_f = (I/2) dx_p: parity 0 -> ON parent point I/2, parity 1
    -> midway between parent points floor(I/2) and floor(I/2) + 1. Brute force by floating-point position."""
    boxes = [wl.Box(0, (0, 0, 0), (24, 24, 24)), wl.Box(1, (10, 12, 14), (20, 18, 16))]
    w = wl.Workload("t", boxes, (24, 24, 24), vertex=1, init=lambda w_, l, ib, c: np.zeros(tuple(reversed(w_.box(l, ib).n))))
    H = oracle_mod.OracleHierarchy.from_workload(w)
    gm = H.ghost_map(1, 0)
    dxp, dxf = w.dx(0), w.dx(1)
    for row in gm[:: max(1, len(gm) // 400)]:
        for a in range(3):
            xf = (boxes[1].lo[a] + row[a]) * dxf
            jp = int(math.floor(xf / dxp + 1e-9))
            par = 0 if abs(xf - jp * dxp) < 1e-12 else 1
            if par:
                assert abs(xf - (jp + 0.5) * dxp) < 1e-12
            assert row[3 + a] == jp - boxes[0].lo[a] and ((row[6] >> a) & 1) == par


@pytest.mark.slow
def test_fd8_ladder_follows_the_stencil_with_matching_interpolation(oracle_mod):
    """cfg-2 (two levels, exact plane wave) at 32^3 to t = 0.5 with 8th-order differences: with the quartic / quintic
    operators the interpolation bounds the composite error; with the 9- / 10-point operators it drops to the level of
    RK4's own time error (the closed form omega t (omega dt)^4 / 120 of a single level: 1.2e-6 at dt = 1/64, t = 1/2)."""
    lo = _plane_errors(oracle_mod, 32, True, fd_order=8, ghost=4, interp=0)
    hi = _plane_errors(oracle_mod, 32, True, fd_order=8, ghost=4, interp=1)
    om = wl.PLANE_OMEGA
    rk4 = om * 0.5 * (om / 64.0) ** 4 / 120.0
    assert max(hi) < 0.35 * max(lo), (lo, hi)
    assert max(hi) < 4.0 * rk4, (hi, rk4)  # measured 3.6e-6 (with the subcycling interface error) against 1.2e-6


@pytest.mark.slow
@pytest.mark.parametrize("sub", [True, False])
def test_vertex_centred_ladder_fourth_order(oracle_mod, sub):
    """Vertex-centred cfg-2: order ~4 against the exact plane wave with 6-point prolongation and injection."""
    e16 = _plane_errors(oracle_mod, 16, sub, vertex=1)
    e32 = _plane_errors(oracle_mod, 32, sub, vertex=1)
    for l in (0, 1):
        assert 3.6 < math.log2(e16[l] / e32[l]) < 4.5, (e16, e32)
