"""Pins for the oracle's CCZ4 + gauge RHS (Eqs. 13-26).

(i)  Flat metric, unit lapse, zero shift: every spacetime RHS component is exactly 0, bit for bit.
(ii) Manufactured exact vacuum solution: Minkowski in wavy coordinates (tests/wavy.py). With KO and
     the kappa dampings off, the oracle RHS of gamma~_ij, A~_ij, chi, K^, Gamma^^i must converge at 4th
     order to the analytic time derivative and d_t Theta -> 0 (Hamiltonian constraint).
(iii) The same with a Killing Z-vector: pins every Theta / Z^i term (kappa_z = 0), d_t Theta != 0.
(iv) Damping terms vanish with the constraints; kappa_c term hand value at one point.
The gauge equations (25)-(26) are pinned by test_oracle_evolution.py (gauge wave speed sqrt(2)).
"""
import math

import numpy as np
import pytest

import wavy
from paper_2510_13965_b200 import synth

NG = 3


def _params(**kw):
    return synth.default_params(**kw)


def test_flat_space_rhs_is_exactly_zero(oracle_mod):
    n = 8
    o = oracle_mod.Oracle(_params(), n, n, n, NG, 0.1)
    U = np.zeros((32,) + o.shape)
    for f in (0, 3, 5, 12, 18):
        U[f] = 1.0
    P = np.zeros((10,) + o.shape)
    P[0], P[7] = 1e-10, 1.0
    K = o.rhs(U, P, "ccz4")
    assert np.all(K[:22] == 0.0)


def _wavy_error(oracle_mod, n, with_Z):
    dx = 2.0 * math.pi / n
    X, Y, Z = synth.mesh(n, n, n, NG, dx)
    t0 = 0.3
    par = _params(kappa_z=0.0, kappa_c=0.0, kappa_2=0.0, sigma_ko_spacetime=0.0, grav_G=0.0)
    o = oracle_mod.Oracle(par, n, n, n, NG, dx)
    U = np.zeros((32,) + o.shape)
    U[:22] = wavy.ccz4_fields(t0, X, Y, Z, with_Z)
    P = np.zeros((10,) + o.shape)
    P[0], P[7] = 1e-10, 1.0
    K = o.rhs(U, P, "ccz4")
    dU = wavy.ddt(lambda t: wavy.ccz4_fields(t, X, Y, Z, with_Z), t0)
    s = (slice(NG, -NG),) * 3
    err = np.array([np.abs(K[f][s] - dU[f][s]).max() for f in range(18)])   # gauge fields are not evolved by (25)-(26) here
    mag = np.array([np.abs(dU[f][s]).max() for f in range(18)])
    return err, mag


@pytest.mark.parametrize("with_Z", [False, True])
def test_wavy_minkowski_exact_solution(oracle_mod, with_Z):
    e1, mag = _wavy_error(oracle_mod, 16, with_Z)
    e2, _ = _wavy_error(oracle_mod, 32, with_Z)
    # every component carries signal (the solution is not trivial) ...
    assert np.all(mag[:14] > 1e-3) and np.all(mag[15:] > 1e-3)
    if with_Z:
        assert mag[14] > 1e-3           # d_t Theta != 0 with the Killing Z-vector
    else:
        assert mag[14] < 1e-10          # d_t Theta = 0: Hamiltonian constraint
    # ... the error is small and falls at 4th order (ratio 16 for halved spacing)
    assert np.all(e2 < 2e-4), e2
    ratio = e1 / e2
    assert np.all(ratio > 11.0) and np.all(ratio < 24.0), ratio


def test_damping_terms(oracle_mod):
    """kappa terms are linear in the constraints: with Theta = 0, Z = 0 (Gamma^ = Gamma~), det gamma~ = 1 and
    A~ trace-free, switching kappa_z, kappa_c on changes nothing beyond truncation-level Z (from FD Gamma~)."""
    n = 16
    dx = 2.0 * math.pi / n
    X, Y, Z = synth.mesh(n, n, n, NG, dx)
    U = np.zeros((32, n + 6, n + 6, n + 6))
    U[:22] = wavy.ccz4_fields(0.3, X, Y, Z, False)
    P = np.zeros((10,) + U.shape[1:])
    P[0], P[7] = 1e-10, 1.0
    base = dict(sigma_ko_spacetime=0.0, grav_G=0.0)
    K0 = oracle_mod.Oracle(_params(kappa_z=0.0, kappa_c=0.0, **base), n, n, n, NG, dx).rhs(U, P, "ccz4")
    K1 = oracle_mod.Oracle(_params(kappa_z=0.7, kappa_c=0.3, kappa_2=0.2, **base), n, n, n, NG, dx).rhs(U, P, "ccz4")
    s = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
    # only Gamma^ sees kappa_z through the O(dx^4) numerical Z^i = chi/2 (Gamma^ - Gamma~_FD)
    assert np.abs(K1[:15][s[1:]] if False else (K1 - K0)[:15][s]).max() < 1e-12
    assert np.abs((K1 - K0)[15:18][s]).max() < 5e-4
    # hand value: uniform state with Theta = th, det gamma~ = d, everything else flat
    th, d = 0.01, 1.3
    U = np.zeros((32, n + 6, n + 6, n + 6))
    U[0], U[3], U[5], U[12], U[18] = d, 1.0, 1.0, 1.0, 1.0
    U[14] = th
    kz, kc, k2 = 0.7, 0.3, 0.2
    K = oracle_mod.Oracle(_params(kappa_z=kz, kappa_c=kc, kappa_2=k2, **base), n, n, n, NG, dx).rhs(U, P, "ccz4")
    c = (n // 2 + NG,) * 3
    # Eq. (13): -alpha/3 kappa_c gamma~_ij ln(det)    (A~ = 0)
    assert K[0][c] == pytest.approx(-kc / 3.0 * d * math.log(d), rel=1e-13)
    assert K[3][c] == pytest.approx(-kc / 3.0 * 1.0 * math.log(d), rel=1e-13)
    # Eq. (15): 2/3 chi alpha (K^ + 2 Theta)
    assert K[12][c] == pytest.approx(2.0 / 3.0 * 2.0 * th, rel=1e-13)
    # Eq. (16): alpha [ (K^+2Theta)^2/3 + kappa_z (1 - kappa_2) Theta ]
    assert K[13][c] == pytest.approx((2 * th) ** 2 / 3.0 + kz * (1 - k2) * th, rel=1e-13)
    # Eq. (17): alpha/2 [ 2/3 Theta (K^ - 2 Theta) ] - alpha kappa_z (2 + kappa_2) Theta
    assert K[14][c] == pytest.approx(0.5 * (2.0 / 3.0 * th * (-2 * th)) - kz * (2 + k2) * th, rel=1e-13)
    # Eq. (25): -2 alpha f K^ = 0 ; Eq. (26): 3/4 f Gamma^ - eta beta = 0
    assert K[18][c] == 0.0 and K[19][c] == 0.0
