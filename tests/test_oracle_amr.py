"""Pins of the oracle's AMR transfer operators: prolongation Eq. (80), copy restriction
(l.626), dense-output interpolators Eqs. (56)-(59) (l.412-434). Everything here is fixed by the paper's printed coefficients or by
mathematics (polynomial exactness, Lagrange remainder, Runge-Kutta order conditions), nothing by the oracle itself."""
import math

import numpy as np
import pytest


def _coarse(fun, n, ng, h, x0=0.0):
    x = x0 + (np.arange(n + 2 * ng) - ng) * h
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    return fun(X, Y, Z)[None].copy()


def test_eq80_printed_coefficients_and_polynomial_exactness(oracle_mod):
    """Impulses return 3, -25, 150, 150, -25, 3 over 256 as printed (l.616); the formula is the Lagrange interpolant through six
    points, so it is exact on polynomials up to degree 5 and not on degree 6. Catches any wrong coefficient or a shifted stencil."""
    L = oracle_mod.lib()
    want = np.array([3, -25, 150, 150, -25, 3]) / 256.0
    for m in range(6):
        u = np.zeros(8)
        u[1 + m] = 1.0                              # u[3] is U_i: offsets -2..3 are u[1..6]
        assert L.orc_prolong_mid(u[3:].ctypes.data, 1) == want[m]
    x = np.arange(-3, 5, dtype=float)
    for deg in range(0, 6):
        u = (x - 0.3) ** deg
        assert abs(L.orc_prolong_mid(u[3:].ctypes.data, 1) - (0.5 - 0.3) ** deg) < 1e-12 * max(1.0, np.abs(u).max())
    u = x ** 6
    assert abs(L.orc_prolong_mid(u[3:].ctypes.data, 1) - 0.5 ** 6) > 1.0


def test_eq80_lagrange_remainder(oracle_mod):
    """f - p = f^(6)(xi)/6! * prod (x - x_j) = -(0.5 * 1.5 * 2.5)^2 h^6 f^(6)/720, so interpolant - exact = +(5/1024) h^6 f^(6):
    sixth order with that constant (a fifth-order / four-point formula fails this)."""
    L = oracle_mod.lib()
    k = 1.3
    errs = []
    for h in (0.2, 0.1, 0.05):
        x = 0.4 + np.arange(-3, 5) * h
        u = np.sin(k * x)
        errs.append(L.orc_prolong_mid(u[3:].ctypes.data, 1) - math.sin(k * (0.4 + 0.5 * h)))
        f6 = -k ** 6 * math.sin(k * (0.4 + 0.5 * h))
        assert errs[-1] == pytest.approx(5.0 / 1024.0 * h ** 6 * f6, rel=0.05)
    assert math.log2(abs(errs[0] / errs[1])) > 5.8


def test_prolongation_3d_tensor_product(oracle_mod):
    """Fine points of a 3-D patch pair: coincident points are copies (bit for bit), every other point is exact for a polynomial of
    degree 5 in each variable (x^5 y^5 z^5 terms included), whatever the parity combination; origin and ghost indices honoured.
    Catches a swapped axis, a wrong origin / parity for negative (ghost) indices and a missing cross term."""
    nc, ngc, nf, ngf = 12, 3, 8, 3
    h = 0.1
    org = (3, 4, 2)
    fun = lambda X, Y, Z: (1 + X + 0.5 * X ** 5) * (2 - Y + Y ** 4 - 0.3 * Y ** 5) * (1 + 0.2 * Z ** 3 + Z ** 5)
    Uc = _coarse(fun, nc, ngc, h)
    Uf = np.full((1, nf + 2 * ngf,) * 1 + (nf + 2 * ngf, nf + 2 * ngf), np.nan)
    oracle_mod.prolong(Uc, ngc, Uf, ngf, org, (0, 0, 0), (nf + 2 * ngf,) * 3)
    xf = [org[d] * h + (np.arange(nf + 2 * ngf) - ngf) * h / 2 for d in range(3)]
    Z, Y, X = np.meshgrid(xf[2], xf[1], xf[0], indexing="ij")
    exact = fun(X, Y, Z)
    assert np.abs(Uf[0] - exact).max() < 1e-12 * np.abs(exact).max()
    # coincident points (all three fine interior indices even): copies
    ev = slice(ngf % 2, None, 2) if ngf % 2 == 0 else slice(1, None, 2)     # array index with even interior index
    sub = Uf[0][ev, ev, ev]
    i0 = [org[d] + ngc + (np.arange(nf + 2 * ngf)[ev] - ngf) // 2 for d in range(3)]
    assert np.array_equal(sub, Uc[0][np.ix_(i0[2], i0[1], i0[0])])
    # a sub-box only: nothing outside it is touched
    Uf2 = np.full_like(Uf, -7.0)
    oracle_mod.prolong(Uc, ngc, Uf2, ngf, org, (0, 2, 5), (3, 9, 14))
    mask = np.zeros(Uf2.shape[1:], bool)
    mask[5:14, 2:9, 0:3] = True
    assert np.array_equal(Uf2[0][mask], Uf[0][mask]) and np.all(Uf2[0][~mask] == -7.0)


def test_restriction_is_a_copy_and_inverts_prolongation(oracle_mod):
    """Restriction copies fine (2i, 2j, 2k) to coarse origin + (i, j, k) and touches nothing else (l.626); restriction after
    prolongation returns the coarse data bit for bit."""
    rng = np.random.default_rng(3)
    nc, ngc, nf, ngf = 12, 3, 9, 3                   # odd fine size: the last even point is index 8
    org = (2, 3, 4)
    Uc = rng.standard_normal((2, nc + 6, nc + 6, nc + 6))
    Uf = rng.standard_normal((2, nf + 6, nf + 6, nf + 6))
    Uc2 = Uc.copy()
    oracle_mod.restrict(Uf, ngf, Uc2, ngc, org)
    want = Uc.copy()
    for k in range(0, nf, 2):
        for j in range(0, nf, 2):
            for i in range(0, nf, 2):
                want[:, org[2] + k // 2 + ngc, org[1] + j // 2 + ngc, org[0] + i // 2 + ngc] = Uf[:, k + ngf, j + ngf, i + ngf]
    assert np.array_equal(Uc2, want)
    Uf3 = np.zeros_like(Uf)
    oracle_mod.prolong(Uc, ngc, Uf3, ngf, org, (0, 0, 0), (nf + 6,) * 3)
    Uc3 = np.zeros_like(Uc)
    oracle_mod.restrict(Uf3, ngf, Uc3, ngc, org)
    sl = (slice(None), slice(org[2] + ngc, org[2] + ngc + 5), slice(org[1] + ngc, org[1] + ngc + 5), slice(org[0] + ngc, org[0] + ngc + 5))
    assert np.array_equal(Uc3[sl], Uc[sl])


@pytest.mark.parametrize("scheme,name", [(0, "rk4"), (1, "ssprk3")])
def test_dense_output_order_conditions(oracle_mod, scheme, name):
    """b_j(theta) of Eqs. (58)-(59) against the Runge-Kutta order conditions of a continuous extension (Hairer-Norsett-Wanner II.6):
    sum b_j = theta, sum b_j c_j = theta^2/2 (order 2) and, for RK4, sum b_j c_j^2 = theta^3/3, sum b_j a_jk c_k = theta^3/6
    (order 3); theta = 1 gives the scheme's weights, theta = 0 gives zero. The derivative option (Eq. 57) against numerical
    differentiation. Catches every coefficient of Eqs. (58)-(59)."""
    from paper_2510_13965_b200 import synth
    a, w = synth.tableau(name)
    c = a.sum(axis=1)
    for th in (0.0, 0.25, 0.5, 0.8, 1.0):
        b = oracle_mod.dense_weights(scheme, th)
        assert b.sum() == pytest.approx(th, abs=1e-15)
        assert b @ c == pytest.approx(th ** 2 / 2, abs=1e-15)
        if scheme == 0:
            assert b @ c ** 2 == pytest.approx(th ** 3 / 3, abs=1e-15)
            assert b @ (a @ c) == pytest.approx(th ** 3 / 6, abs=1e-15)
    assert np.allclose(oracle_mod.dense_weights(scheme, 1.0), w, atol=1e-15)
    for m in (1, 2, 3):
        th, e = 0.6, 1e-3
        num = oracle_mod.dense_weights(scheme, th, m - 1)
        num = (oracle_mod.dense_weights(scheme, th + e, m - 1) - oracle_mod.dense_weights(scheme, th - e, m - 1)) / (2 * e)
        assert np.allclose(oracle_mod.dense_weights(scheme, th, m), num, atol=1e-5)


def test_dense_output_interpolates_an_ode_to_its_order(oracle_mod):
    """y' = lambda y through the patch routine: RK4 stages K_j = F(U^(j)) built by hand, dense output at theta vs exp(lambda theta dt):
    error O(dt^4) for Eq. (58) (third-order interpolant) — halving dt divides it by ~16; first derivative (Eq. 57) O(dt^3)."""
    lam = -0.7
    errs, derrs = [], []
    o = oracle_mod.Oracle(dict(), 2, 2, 2, 3, 1.0)
    for dt in (0.4, 0.2):
        y0 = np.full((1, 8, 8, 8), 1.3)
        k1 = lam * y0
        k2 = lam * (y0 + 0.5 * dt * k1)
        k3 = lam * (y0 + 0.5 * dt * k2)
        k4 = lam * (y0 + dt * k3)
        th = 0.37
        y = o.dense_output(y0, [k1, k2, k3, k4], 0, th, dt)
        errs.append(abs(y[0, 4, 4, 4] - 1.3 * math.exp(lam * th * dt)))
        assert y[0, 0, 0, 0] == 1.3                                      # ghosts are not touched
        dy = o.dense_output(y0, [k1, k2, k3, k4], 0, th, dt, deriv=1)
        derrs.append(abs(dy[0, 4, 4, 4] - 1.3 * lam * math.exp(lam * th * dt)))
    assert 12 < errs[0] / errs[1] < 20, errs
    assert 6 < derrs[0] / derrs[1] < 10, derrs
