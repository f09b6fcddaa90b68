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


# ---- WENO5 (refs. [61], [63]) -------------------------------------------------------
def _weno(oracle, f, eps=1e-6):
    return oracle.lib().orc_weno5(*[float(x) for x in f], float(eps))


def test_weno5_linear_weights_give_eq70(oracle_mod):
    """With epsilon >> IS_k the non-linear weights are the linear ones and the scheme must be the fifth-order formula the paper
    prints as Eq. (70), (2, -13, 47, 27, -3)/60. Catches a wrong candidate coefficient or a wrong / permuted linear weight."""
    rng = np.random.default_rng(5)
    for _ in range(20):
        f = rng.uniform(-1, 1, 5)
        want = (2 * f[0] - 13 * f[1] + 47 * f[2] + 27 * f[3] - 3 * f[4]) / 60.0
        assert abs(_weno(oracle_mod, f, eps=1e30) - want) < 1e-14


def test_weno5_smoothness_indicators_from_their_definition(oracle_mod):
    """IS_k = sum_{l=1,2} int_cell h^(2l-1) (d^l p_k / dx^l)^2 dx for the parabola p_k whose cell averages match the three
    stencil values ([63] Eq. 3.1): computed here with numpy polynomials, independently of the closed forms 13/12 (..)^2 +
    1/4 (..)^2 in the oracle; the weights rebuilt from it must reproduce the oracle's value. Catches a wrong 13/12, 1/4 or
    a wrong difference inside either square."""
    from numpy.polynomial import polynomial as Pn
    rng = np.random.default_rng(6)

    def indicator(vals, offs):                      # cells centred at offs (h = 1), target cell centred at 0
        A = np.array([[((o + 0.5) ** (m + 1) - (o - 0.5) ** (m + 1)) / (m + 1) for m in range(3)] for o in offs])
        c = np.linalg.solve(A, vals)                # p(x) = c0 + c1 x + c2 x^2 with matching cell averages
        d1, d2 = Pn.polyder(c, 1), Pn.polyder(c, 2)
        I1 = Pn.polyint(Pn.polymul(d1, d1))
        I2 = Pn.polyint(Pn.polymul(d2, d2))
        return (Pn.polyval(0.5, I1) - Pn.polyval(-0.5, I1)) + (Pn.polyval(0.5, I2) - Pn.polyval(-0.5, I2)), Pn.polyval(0.5, c)

    for eps in (1e-6, 1e-12):
        for _ in range(20):
            f = rng.uniform(-1, 1, 5)
            parts = [indicator(f[0:3], (-2, -1, 0)), indicator(f[1:4], (-1, 0, 1)), indicator(f[2:5], (0, 1, 2))]
            al = np.array([d / (eps + b) ** 2 for d, (b, _) in zip((0.1, 0.6, 0.3), parts)])
            want = float((al * np.array([q for _, q in parts])).sum() / al.sum())
            assert abs(_weno(oracle_mod, f, eps) - want) < 1e-12 * max(1.0, abs(want)), (f, eps)


def test_weno5_order_and_eno_property(oracle_mod):
    """Fifth-order convergence of the reconstructed interface value on smooth cell averages; on a step the value stays within the
    data range to O(eps) (essentially non-oscillatory: the stencils that cross the step get vanishing weight)."""
    errs = []
    for n in (128, 256, 512):                                                                           # (the Jiang-Shu weights approach the linear ones only as O(h^2): pre-asymptotic below)
        h = 1.0 / n
        xs = (np.arange(-2, 3)) * h + 0.3 - h / 2                                                       # the interface sits at x = 0.3
        avg = (np.cos(2 * np.pi * (xs - h / 2)) - np.cos(2 * np.pi * (xs + h / 2))) / (2 * np.pi * h)   # cell averages of sin(2 pi x)
        errs.append(abs(_weno(oracle_mod, avg) - np.sin(2 * np.pi * 0.3)))
    assert np.log2(errs[0] / errs[1]) > 4.6 and np.log2(errs[1] / errs[2]) > 4.6, errs
    for f in ([0, 0, 0, 1, 1], [0, 0, 1, 1, 1], [1, 1, 1, 0, 0], [0, 1, 1, 1, 1], [3, 3, -2, -2, -2]):
        v = _weno(oracle_mod, f)
        assert min(f) - 1e-5 <= v <= max(f) + 1e-5, (f, v)


def test_weno5_selected_by_recon_kind(oracle_mod):
    """rhs_grmhd with recon_kind = 1 differs from MP5 only through R of Eq. (66): with linear weights (huge epsilon) WENO5 is Eq. (70),
    which MP5 returns wherever the test of Eq. (72) passes, so the two flux divergences agree to rounding at most points of a
    smooth state (and differ where MP5 limits); with the standard epsilon they differ by the weights' O(h^2) departure."""
    from paper_2510_13965_b200 import synth
    cfg = synth.config1(n=12)
    out = {}
    for name, kind, eps in (("mp5", 0, 1e-6), ("lin", 1, 1e30), ("weno", 1, 1e-6)):
        par = dict(cfg["params"], recon_kind=kind, weno_eps=eps)
        o = oracle_mod.Oracle(par, 12, 12, 12, 3, cfg["dx"])
        U, P = cfg["U"].copy(), cfg["P"].copy()
        o.prim2con(U, P)
        o.fill_ghosts(U, cfg["bc"])
        Pq, _ = o.con2prim(U)
        out[name] = o.rhs(U, Pq, part="grmhd_flux")[22:, 3:-3, 3:-3, 3:-3]
    scale = np.abs(out["mp5"]).reshape(10, -1).max(axis=1)[:, None, None, None]
    same = np.abs(out["lin"] - out["mp5"]) < 1e-11 * scale
    assert 0.3 < same.mean() < 1.0, same.mean()
    assert np.abs(out["weno"] - out["lin"]).max() > 1e-8 * scale.max()
