"""Oracle pins that need time evolution (BASELINE.json north_star): observed convergence order on the
linearised gauge wave and the circularly polarised Alfven wave, TOV equilibrium, monotone Riemann problem.
All 1-D problems run on thin slabs (n x 4 x 4, periodic across) so the whole file takes about a minute on one core."""
import math

import numpy as np
import pytest

from paper_2510_13965_b200 import synth

NG = 3
I = (slice(NG, -NG),) * 3


def _evolve(oracle_mod, cfg, t_end, courant=0.25, rk="rk4"):
    n = cfg["n"]
    o = oracle_mod.Oracle(cfg["params"], n[0], n[1], n[2], cfg["ng"], cfg["dx"], table=cfg.get("table"))
    U, P = cfg["U"].copy(), cfg["P"].copy()
    o.prim2con(U, P)
    a, w = synth.tableau(rk)
    steps = int(round(t_end / (courant * cfg["dx"])))
    dt = t_end / steps
    Pf, F = o.evolve(U, cfg["bc"], a, w, dt, steps)
    return U, Pf, F


def test_gauge_wave_speed_and_fourth_order(oracle_mod):
    """Eqs. (16), (25): alpha = 1 + A sin k(x - sqrt2 t) solves the linearised system; the centred stencils are 4th order."""
    t_end, err = 0.25, {}
    for n in (16, 32):
        cfg = synth.config2_gauge_wave(n=n, ny=4)
        U, _, _ = _evolve(oracle_mod, cfg, t_end)
        al, Kh = cfg["exact"](t_end)
        err[n] = (np.abs(U[synth.ALPHA] - al)[I].max(), np.abs(U[synth.KHAT] - Kh)[I].max())
        # a wrong speed (e.g. 1 instead of sqrt 2) would leave an O(A) = 1e-6 error
        assert err[n][0] < 2e-9 and err[n][1] < 2e-8, err
    order = math.log2(err[16][0] / err[32][0])
    assert 3.5 < order < 5.0, (order, err)
    # the metric stays flat and the shift zero to round-off (linearised solution, f_beta = eta = 0)
    assert np.abs(U[synth.BETAX:synth.BETAX + 3]).max() == 0.0


def test_alfven_wave_convergence(oracle_mod):
    """Exact SRMHD solution run through the coupled RHS with grav_G = 0 (R29): flux brackets of Eq. (32), flux
    splitting + MP5 (5th order in space) and RK4 must converge at >= 4th order; the spacetime stays exactly flat."""
    t_end, err = 0.2, {}
    for n in (16, 32):
        cfg = synth.config2_alfven(n=n, ny=4)
        U, P, F = _evolve(oracle_mod, cfg, t_end)
        ex = cfg["exact"](t_end)
        err[n] = max(np.abs(U[synth.BXBAR + i] - ex["B"][i])[I].max() for i in range(3))
        assert np.all(F == 0)
        flat = synth._flat_state(U.shape[1:])
        assert np.array_equal(U[:22], flat[:22])
    order = math.log2(err[16] / err[32])
    assert err[32] < 2e-4 and order > 3.8, (order, err)


def test_tov_equilibrium(oracle_mod):
    """Config 3 at two resolutions: inside the star the RHS of every field tends to 0 at 4th order (hydrostatic balance
    d_i p = -(rho h) d_i ln alpha from Eq. (32); the matter couplings 4 pi (tau + S), -8 pi S_ij^TF ... of Eqs. (14)-(19))."""
    res = {}
    for n in (24, 48):
        cfg = synth.config3(n=n, half_width=9.0, b_scale=0.0)
        o = oracle_mod.Oracle(cfg["params"], n, n, n, cfg["ng"], cfg["dx"])
        U, P = cfg["U"].copy(), cfg["P"].copy()
        o.prim2con(U, P)
        Pc, F = o.con2prim(U)
        K = o.rhs(U, Pc)
        X, Y, Z = synth.mesh(n, n, n, cfg["ng"], cfg["dx"], x0=(-9.0 + 0.5 * cfg["dx"],) * 3)
        core = (np.sqrt(X * X + Y * Y + Z * Z) < 0.55 * cfg["tov"]["Rbar"])[I]
        res[n] = {f: np.abs(K[f][I][core]).max() for f in (synth.KHAT, synth.AXX, synth.GAMX, synth.SXBAR, synth.TAUBAR, synth.ALPHA)}
    # scales: d_x p ~ 1e-5, 4 pi (tau + S) alpha ~ 1e-2
    assert res[48][synth.SXBAR] < 3e-9 and res[48][synth.KHAT] < 2e-6, res
    for f in (synth.KHAT, synth.SXBAR, synth.AXX):
        assert res[24][f] / res[48][f] > 10.0, (f, res)
    assert res[48][synth.ALPHA] < 1e-7 and res[48][synth.TAUBAR] < 1e-7     # O(h^5) dissipation only: Kreiss-Oliger (alpha), Lax-Friedrichs splitting (tau)


def test_tov_short_run_holds(oracle_mod):
    cfg = synth.config3(n=24, half_width=12.0)
    rho0 = cfg["P"][synth.RHO].max()
    U, P, F = _evolve(oracle_mod, cfg, 5 * 0.25 * cfg["dx"])
    assert abs(P[synth.RHO].max() / rho0 - 1.0) < 2e-3
    assert (F & 32).sum() == 0 and (F & 64).sum() == 0           # nothing fatal, every solve converged
    assert (F & 1).sum() > 0.5 * F.size                           # the atmosphere is flagged as such


def test_riemann_problem_stays_monotone(oracle_mod):
    """1-D magnetised shock tube (Brio-Wu / Balsara-1 states): no spurious over/undershoots from the flux-splitting +
    MP5 limiter (Eqs. 65-76). The exact solution itself is not monotone (compound wave, contact, and a right fast
    rarefaction that lowers rho to ~0.115), so the pin is: rho stays inside the range of the exact wave fan and the total
    variation stays at that of the fan (~1.16) plus a small allowance, instead of growing with Gibbs oscillations."""
    cfg = synth.riemann_1d(n=128, ny=4)
    U, P, F = _evolve(oracle_mod, cfg, 0.2, courant=0.25)
    rho = P[synth.RHO][NG, NG, NG:-NG]
    assert rho.max() < 1.0 + 1e-3 and rho.min() > 0.105, (rho.max(), rho.min())
    tv = np.abs(np.diff(rho)).sum()
    assert tv < 1.35, tv
    assert (F & (32 | 64)).sum() == 0
    assert np.abs(np.diff(rho)).max() < 0.5                       # the initial jump has spread into the wave fan
