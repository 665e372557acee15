"""Pins for the oracle's dense output (eqs 10-18). CPU only."""
import os
from fractions import Fraction

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _frac(s):
    return float(Fraction(s))


def test_b_invariants(oracle_mod):
    o = oracle_mod
    # theta = 0 returns y_n; theta = 1 reproduces the RK4 weights of eq (5)
    for i in range(1, 5):
        assert o.b(i, 0, 0.0) == 0.0
    assert np.allclose([o.b(i, 0, 1.0) for i in range(1, 5)], [1 / 6, 1 / 3, 1 / 3, 1 / 6], rtol=0, atol=1e-16)
    # order conditions of a 3rd-order continuous extension of RK4 (c = 0, 1/2, 1/2, 1; a21=a32=1/2, a43=1)
    c = np.array([0.0, 0.5, 0.5, 1.0])
    a = np.zeros((4, 4))
    a[1, 0] = a[2, 1] = 0.5
    a[3, 2] = 1.0
    for th in np.linspace(0, 1, 11):
        bb = np.array([o.b(i, 0, th) for i in range(1, 5)])
        assert abs(bb.sum() - th) < 1e-15
        assert abs(bb @ c - th ** 2 / 2) < 1e-15
        assert abs(bb @ c ** 2 - th ** 3 / 3) < 1e-15
        assert abs(bb @ (a @ c) - th ** 3 / 6) < 1e-15


def test_b_derivatives_by_finite_difference(oracle_mod):
    o = oracle_mod
    e = 1e-4
    for i in range(1, 5):
        for th in (0.0, 0.3, 0.5, 0.9):
            for m in (1, 2, 3):
                fd = (o.b(i, m - 1, th + e) - o.b(i, m - 1, th - e)) / (2 * e)
                assert abs(fd - o.b(i, m, th)) < 1e-7, (i, m, th)


def test_folded_coefficient_table(oracle_mod):
    """Direct evaluation of eqs (10),(14)-(18) at unit k vectors equals the rational table."""
    o = oracle_mod
    rows = [l.split() for l in open(os.path.join(GOLD, "dense_coeffs.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 10
    for r in rows:
        stage, theta = int(r[0]), _frac(r[1])
        want = [_frac(x) for x in r[2:6]]
        for hp in (1.0, 0.37):
            got = [o.dense_stage(stage, theta, hp, 0.0, np.eye(4)[m]) / hp for m in range(4)]
            assert np.allclose(got, want, rtol=0, atol=4e-16), (stage, theta, got, want)
        # y_old passes through with weight one
        assert o.dense_stage(stage, theta, 0.5, 1.25, np.zeros(4)) == 1.25


def test_theta_one_reproduces_rk4_update(oracle_mod):
    o = oracle_mod
    rng = np.random.default_rng(1)
    for _ in range(20):
        y0, h = rng.normal(), rng.uniform(0.01, 1.0)
        k = rng.normal(size=4)
        want = y0 + h / 6 * (k[0] + 2 * k[1] + 2 * k[2] + k[3])
        got = o.dense_stage(5, 1.0, h, y0, k)
        assert abs(got - want) <= 4e-16 * max(1.0, abs(want))
        assert o.dense_stage(1, 0.0, h, y0, k) == y0


def _f(y):
    return -y * y + np.sin(y)


def _rk4_slopes(y0, h):
    k1 = _f(y0)
    k2 = _f(y0 + h / 2 * k1)
    k3 = _f(y0 + h / 2 * k2)
    k4 = _f(y0 + h * k3)
    return np.array([k1, k2, k3, k4])


@pytest.mark.parametrize("theta", [0.0, 0.5])
def test_ghost_stage_order_scalar_ode(oracle_mod, theta):
    """Eqs (15)-(18) with the PARENT step in f_y y'' (reading S5) give ghost stage vectors that agree
    with the child's own RK4 stages (started from the dense-output value) to O(h^4): the error falls by
    >= ~16 per halving. SURVEY.md Appendix A quotes, for theta = 0 and h_p = 0.1, 0.05, 0.025:
    Y_3: 3.6e-9, 1.2e-10, 4.1e-12; Y_4: 5.4e-8, 3.2e-9, 1.9e-10."""
    o = oracle_mod
    y0 = 0.7
    errs = {2: [], 3: [], 4: []}
    for hp in (0.1, 0.05, 0.025):
        k = _rk4_slopes(y0, hp)
        ys = o.dense_stage(1, theta, hp, y0, k)
        h = hp / 2
        Y2 = ys + h / 2 * _f(ys)
        Y3 = ys + h / 2 * _f(Y2)
        Y4 = ys + h * _f(Y3)
        for s, true in ((2, Y2), (3, Y3), (4, Y4)):
            errs[s].append(abs(o.dense_stage(s, theta, hp, y0, k) - true))
    for s in (2, 3, 4):
        e = errs[s]
        if max(e) < 1e-15:  # Y_2 at theta = 0 is exact: y' = k_1 = f(y_n)
            continue
        assert e[0] / e[1] > 12 and e[1] / e[2] > 12, (s, e)
    if theta == 0.0:
        assert np.allclose(errs[3], [3.6e-9, 1.2e-10, 4.1e-12], rtol=0.08)
        assert np.allclose(errs[4], [5.4e-8, 3.2e-9, 1.9e-10], rtol=0.08)


def test_dense_output_accuracy_scalar_ode(oracle_mod):
    """Eq (10): y(t_n + theta h) to O(h^4) locally — compare with a tight reference solution."""
    o = oracle_mod
    y0 = 0.7

    def ref(t):  # RK4 with 2000 tiny steps
        n = 2000
        y, h = y0, t / n
        for _ in range(n):
            k = _rk4_slopes(y, h)
            y = y + h / 6 * (k[0] + 2 * k[1] + 2 * k[2] + k[3])
        return y

    for th in (0.25, 0.5, 0.75):
        e = []
        for hp in (0.2, 0.1, 0.05):
            k = _rk4_slopes(y0, hp)
            e.append(abs(o.dense_stage(5, th, hp, y0, k) - ref(th * hp)))
        assert e[0] / e[1] > 12 and e[1] / e[2] > 12, (th, e)
