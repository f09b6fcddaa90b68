"""Pins for the oracle's GRMHD fluxes, sources and flux-splitting discretisation (Eq. 32, Sec. III C).

(i)   Uniform boosted magnetised fluid in wavy-Minkowski coordinates (tests/wavy.py): exact solution of
      nabla.T = 0, nabla.*F = 0. The oracle's RHS for Dbar, DYebar, taubar, Sbar_i, Bbar^i must converge to the
      analytic time derivative of the conserved fields (>= 4th order: sources use Eq. 60) and the phibar RHS
      (= -d_k(alpha c_b^2 Bbar^k) + ...) must converge to 0 (solenoidal field, phi = 0).
(ii)  Flat space, uniform state: RHS is exactly 0 (flux-sum consistency F^(U const) = F, Eq. 69).
(iii) Flat-space limit of the cleaning subsystem = Dedner telegraph system: d_t phi = -c_b^2 div B - kappa_b phi,
      d_t B^i = -d_i phi for a fluid at rest.
"""
import math

import numpy as np
import pytest

import wavy
from paper_2510_13965_b200 import synth

NG = 3
S = (slice(NG, -NG),) * 3


def _state(oracle_mod, o, t, X, Y, Z):
    a, v, W, B = wavy.fluid(t, X, Y, Z)
    U = np.zeros((32,) + X.shape)
    U[:22] = synth.conformal_from_adm(a["gam"], a["dgam"], a["Kij"], a["alpha"], a["beta"])
    sg = np.sqrt(a["det"])
    for i in range(3):
        U[synth.BXBAR + i] = sg * B[i]
    P = np.zeros((10,) + X.shape)
    P[synth.RHO], P[synth.YE], P[synth.EPS] = wavy.RHO0, 0.25, wavy.EPS0
    for i in range(3):
        P[synth.VX + i] = v[i]
    o.prim2con(U, P)
    assert np.allclose(P[synth.WLOR], W, rtol=1e-12)      # W from the 3-velocity agrees with alpha u^t
    return U, P


def _wavy_fluid_error(oracle_mod, n):
    dx = 2.0 * math.pi / n
    X, Y, Z = synth.mesh(n, n, n, NG, dx)
    par = synth.default_params(grav_G=0.0, eos_gamma=5.0 / 3.0, c_b=0.8, kappa_b=0.7)
    o = oracle_mod.Oracle(par, n, n, n, NG, dx)
    t0 = 0.3
    U, P = _state(oracle_mod, o, t0, X, Y, Z)
    K = o.rhs(U, P, "grmhd")
    dU = wavy.ddt(lambda t: _state(oracle_mod, o, t, X, Y, Z)[0], t0)
    # L1 norms for the order (the MP5 limiter clips a handful of isolated smooth extrema by a relative ~3e-7 of
    # the flux, which shows up as single-point spikes in the max norm but not in the L1 norm), max norm as a bound
    err = np.array([np.abs(K[f][S] - dU[f][S]).mean() for f in range(22, 32)])
    emax = np.array([np.abs(K[f][S] - dU[f][S]).max() for f in range(22, 32)])
    mag = np.array([np.abs(dU[f][S]).max() for f in range(22, 32)])
    return err, emax, mag


def test_boosted_fluid_in_wavy_minkowski(oracle_mod):
    e1, _, mag = _wavy_fluid_error(oracle_mod, 16)
    e2, emax2, _ = _wavy_fluid_error(oracle_mod, 32)
    assert np.all(mag[:9] > 1e-6), mag                    # non-trivial evolution of every conserved field
    assert mag[9] < 1e-12                                 # phi stays 0 in the exact solution
    assert np.all(emax2[:9] / mag[:9] < 5e-3), emax2[:9] / mag[:9]
    assert np.all(e2[:9] / mag[:9] < 2e-4), e2[:9] / mag[:9]
    assert emax2[9] < 1e-6                                # -alpha c_b^2 d_k Bbar^k -> 0
    ratio = e1 / e2
    assert np.all(ratio > 12.0), ratio                    # >= 4th order (sources Eq. 60; fluxes 5th, Eq. 70)


def test_uniform_state_flat_space_zero_rhs(oracle_mod):
    n = 8
    o = oracle_mod.Oracle(synth.default_params(), n, n, n, NG, 0.1)
    U = np.zeros((32,) + o.shape)
    for f in (0, 3, 5, 12, 18):
        U[f] = 1.0
    U[28], U[29], U[30] = 0.01, -0.02, 0.03
    P = np.zeros((10,) + o.shape)
    P[0], P[1], P[2] = 1e-3, 0.3, 0.1
    P[4], P[5], P[6] = 0.2, -0.1, 0.3
    o.prim2con(U, P)
    K = o.rhs(U, P, "grmhd")
    scale = np.abs(U[22:32]).max()
    assert np.abs(K[22:32][(slice(None),) + S]).max() < 1e-13 * scale / 0.1


def test_dedner_limit(oracle_mod):
    n = 32
    dx = 2.0 * math.pi / n
    X, Y, Z = synth.mesh(n, n, n, NG, dx)
    cb, kb = 0.8, 0.7
    o = oracle_mod.Oracle(synth.default_params(c_b=cb, kappa_b=kb, grav_G=0.0), n, n, n, NG, dx)
    U = np.zeros((32,) + X.shape)
    for f in (0, 3, 5, 12, 18):
        U[f] = 1.0
    amp = 1e-4
    U[28] = amp * np.sin(X + 2 * Y)                        # div B = amp cos(x + 2y)
    U[29] = amp * np.cos(Z)
    U[31] = amp * np.sin(2 * X - Z)                        # phi
    P = np.zeros((10,) + X.shape)
    P[0], P[1], P[2] = 1.0, 0.3, 0.1                       # heavy fluid at rest: B does not move it at O(amp)
    o.prim2con(U, P)
    K = o.rhs(U, P, "grmhd")
    dphi = -cb * cb * amp * np.cos(X + 2 * Y) - kb * U[31]
    assert np.abs(K[31][S] - dphi[S]).max() < 2e-3 * amp
    gradphi = [amp * 2 * np.cos(2 * X - Z), 0 * X, -amp * np.cos(2 * X - Z)]
    for i in range(3):
        assert np.abs(K[28 + i][S] + gradphi[i][S]).max() < 2e-3 * amp
