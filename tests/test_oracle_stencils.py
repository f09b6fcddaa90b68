"""Pins for the oracle's finite-difference stencils (Sec. III B, Eqs. 60-62, l.454-460).

Pins: exactness on polynomials up to degree 4 (what "fourth order" means), the leading error
constants obtained from the printed coefficients by Taylor expansion
(D1: -h^4 u^(5)/30, D2: -h^4 u^(6)/90, advective: +h^4 u^(5)/20 [beta>0] , KO: sigma h^5 u^(6)/64),
and the printed coefficients themselves applied to a unit impulse.
"""
import math

import numpy as np
import pytest


def line(fun, h, r=3):
    x = np.arange(-r, r + 1) * h
    return fun(x)


@pytest.mark.parametrize("deg", range(0, 5))
def test_d1_d2_adv_exact_on_polynomials(oracle_mod, deg):
    h = 0.37
    x0 = 0.9
    f = lambda x: (x + x0) ** deg
    u = line(f, h)
    d1_exact = deg * x0 ** (deg - 1) if deg > 0 else 0.0
    d2_exact = deg * (deg - 1) * x0 ** (deg - 2) if deg > 1 else 0.0
    assert oracle_mod.stencil("d1", u, 1, h) == pytest.approx(d1_exact, abs=1e-13)
    assert oracle_mod.stencil("d2", u, 1, h) == pytest.approx(d2_exact, abs=1e-12)
    assert oracle_mod.stencil("dadv", u, 1, h, +1.0) == pytest.approx(d1_exact, abs=1e-12)
    assert oracle_mod.stencil("dadv", u, 1, h, -1.0) == pytest.approx(d1_exact, abs=1e-12)
    assert oracle_mod.stencil("dadv", u, 1, h, 0.0) == oracle_mod.stencil("dadv", u, 1, h, 1.0)  # R15
    # KO annihilates polynomials up to degree 5
    assert oracle_mod.stencil("dko", u, 1, h, 0.1) == pytest.approx(0.0, abs=1e-12)


def test_leading_error_constants(oracle_mod):
    h = 0.5
    # u = x^5: u^(5) = 120 ; u = x^6: u^(6) = 720 (evaluated at x = 0, lower derivatives vanish there)
    u5 = line(lambda x: x ** 5, h)
    u6 = line(lambda x: x ** 6, h)
    assert oracle_mod.stencil("d1", u5, 1, h) == pytest.approx(-h ** 4 * 120 / 30, rel=1e-12)
    assert oracle_mod.stencil("d2", u6, 1, h) == pytest.approx(-h ** 4 * 720 / 90, rel=1e-12)
    assert oracle_mod.stencil("dadv", u5, 1, h, 1.0) == pytest.approx(+h ** 4 * 120 / 20, rel=1e-12)
    assert oracle_mod.stencil("dadv", u5, 1, h, -1.0) == pytest.approx(+h ** 4 * 120 / 20, rel=1e-12)
    sigma = 0.1
    assert oracle_mod.stencil("dko", u6, 1, h, sigma) == pytest.approx(sigma * h ** 5 * 720 / 64, rel=1e-12)


def test_printed_coefficients_on_impulses(oracle_mod):
    """Apply each stencil to unit impulses: reproduces the coefficient lists printed in PAPER.md:439-460."""
    h = 1.0
    printed = {
        "d1": ([0, 1, -8, 0, 8, -1, 0], 12.0, ()),
        "d2": ([0, -1, 16, -30, 16, -1, 0], 12.0, ()),
        "dadv_neg": ([-1, 6, -18, 10, 3, 0, 0], 12.0, (-1.0,)),
        "dadv_pos": ([0, 0, -3, -10, 18, -6, 1], 12.0, (1.0,)),
        "dko": ([1, -6, 15, -20, 15, -6, 1], 64.0, (1.0,)),
    }
    for name, (coef, den, extra) in printed.items():
        fn = name.split("_")[0]
        for m in range(7):
            u = np.zeros(7)
            u[m] = 1.0
            assert oracle_mod.stencil(fn, u, 1, h, *extra) == pytest.approx(coef[m] / den, abs=1e-15), (name, m)


def test_mixed_derivative(oracle_mod):
    """Eq. (61): D_xy = D_y(D_x); exact on x^a y^b with a,b <= 4; equals the tensor product of Eq. (60) weights."""
    h1, h2 = 0.3, 0.45
    x = (np.arange(-2, 3) * h1)[None, :]
    y = (np.arange(-2, 3) * h2)[:, None]
    x0, y0 = 0.7, -0.4
    for a in range(5):
        for b in range(5):
            u = (x + x0) ** a * (y + y0) ** b
            exact = (a * x0 ** (a - 1) if a else 0.0) * (b * y0 ** (b - 1) if b else 0.0)
            got = oracle_mod.stencil("d11", u, 1, h1, 5, h2)
            assert got == pytest.approx(exact, abs=1e-12), (a, b)
    w = np.array([1, -8, 0, 8, -1]) / 12.0
    rng = np.random.default_rng(0)
    u = rng.standard_normal((5, 5))
    assert oracle_mod.stencil("d11", u, 1, h1, 5, h2) == pytest.approx((w[:, None] * w[None, :] * u).sum() / (h1 * h2), rel=1e-12)


def test_fourth_order_convergence(oracle_mod):
    f = lambda x: np.sin(1.3 * x + 0.2)
    errs = []
    for h in (0.1, 0.05):
        u = line(f, h)
        errs.append(abs(oracle_mod.stencil("d1", u, 1, h) - 1.3 * math.cos(0.2)))
    assert 14.0 < errs[0] / errs[1] < 18.0
