"""Pins of the M1 oracle: closure limits and exactness, App. C forms vs Sec. II C, Jacobian vs finite
differences, implicit-solve limits, flux consistency, IMEX order conditions."""
import math

import numpy as np
import pytest

from paper_2510_13965_b200 import synth

ID = np.eye(3)


def _rand_state(rng, vmax=0.5, metric=True):
    if metric:
        A = ID + 0.2 * rng.standard_normal((3, 3))
        gl = A @ A.T
    else:
        gl = ID.copy()
    gu = np.linalg.inv(gl)
    v = rng.uniform(-1, 1, 3)
    v *= rng.uniform(0.05, vmax) / math.sqrt(v @ gl @ v)
    W = 1.0 / math.sqrt(1.0 - v @ gl @ v)
    E = 10.0 ** rng.uniform(-8, -2)
    F = rng.uniform(-1, 1, 3)
    F *= rng.uniform(0.05, 0.9) * E / math.sqrt(F @ gu @ F)
    return E, F, v, W, gl, gu


def test_closure_limits(oracle_mod):
    E, F0, v0 = 2.5e-3, np.zeros(3), np.zeros(3)
    c = oracle_mod.m1_closure_point(E, F0, v0, 1.0, ID, ID)
    assert c["xi"] == 0.0 and abs(c["chi"] - 1 / 3) < 1e-16 and np.allclose(c["P"], E * ID / 3, rtol=1e-15, atol=0)
    F = np.array([0.6, -0.48, 0.64]) * E                      # |F| = E
    c = oracle_mod.m1_closure_point(E, F, v0, 1.0, ID, ID)
    assert abs(c["xi"] - 1.0) < 1e-12 and abs(c["chi"] - 1.0) < 1e-12
    assert np.allclose(c["P"], E * np.outer(F, F) / (F @ F), rtol=1e-14, atol=0)


def test_closure_exact_in_thick_and_thin_limits(oracle_mod):
    """Minerbo is exact for radiation isotropic in the fluid frame and for a single beam: build T^ab in flat
    space from its definition, project with n^a, feed (E, F_i) to the closure and compare J, H, P_ij."""
    rng = np.random.default_rng(1)
    for _ in range(20):
        v = rng.uniform(-0.5, 0.5, 3)
        W = 1.0 / math.sqrt(1.0 - v @ v)
        J0 = 10.0 ** rng.uniform(-6, -2)
        E = 4 / 3 * J0 * W * W - J0 / 3
        F = 4 / 3 * J0 * W * W * v
        Pex = 4 / 3 * J0 * W * W * np.outer(v, v) + J0 / 3 * ID
        c = oracle_mod.m1_closure_point(E, F, v, W, ID, ID)
        assert c["xi"] < 1e-7 and abs(c["J"] / J0 - 1) < 1e-12 and np.abs(c["H"]).max() < 1e-12 * J0
        assert np.abs(c["P"] - Pex).max() < 1e-12 * E
        k = rng.standard_normal(3)
        k /= np.linalg.norm(k)
        Eb = 10.0 ** rng.uniform(-6, -2)
        c = oracle_mod.m1_closure_point(Eb, Eb * k, v, W, ID, ID)
        assert abs(c["xi"] - 1.0) < 1e-7 and np.abs(c["P"] - Eb * np.outer(k, k)).max() < 1e-7 * Eb
        assert abs(c["J"] / (W * W * Eb * (1 - k @ v) ** 2) - 1) < 1e-12


def test_closure_orthogonality_and_root(oracle_mod):
    """H^a u_a = 0 (i.e. H.n + H_i v^i = 0) pins the mutual consistency of Eqs. (42)-(44); xi^2 J^2 = H_a H^a at the root."""
    rng = np.random.default_rng(2)
    for _ in range(50):
        E, F, v, W, gl, gu = _rand_state(rng)
        c = oracle_mod.m1_closure_point(E, F, v, W, gl, gu)
        assert abs(c["Hn"] + c["H"] @ v) < 1e-13 * E
        H2 = -c["Hn"] ** 2 + c["H"] @ gu @ c["H"]
        assert 0.0 < c["xi"] < 1.0 and abs(c["xi"] ** 2 * c["J"] ** 2 - H2) < 1e-12 * E * E
        assert abs(c["chi"] - (1 / 3 + c["xi"] ** 2 * (6 - 2 * c["xi"] + 6 * c["xi"] ** 2) / 15)) < 1e-15
        assert np.allclose(c["P"], c["P"].T, rtol=0, atol=1e-18)


def test_appC_forms_equal_section2C(oracle_mod):
    rng = np.random.default_rng(3)
    for _ in range(50):
        E, F, v, W, gl, gu = _rand_state(rng)
        c = oracle_mod.m1_closure_point(E, F, v, W, gl, gu)
        dthin, dthick = 0.5 * (3 * c["chi"] - 1), 1.5 * (1 - c["chi"])
        J, H = oracle_mod.m1_JH(E, F, v, W, gl, gu, dthin, dthick)
        assert abs(J / c["J"] - 1) < 1e-12 and np.abs(H - c["H"]).max() < 1e-12 * E


def _RV(oracle_mod, V, v, W, gl, gu, dthin, dthick, alpha, ka, ks, eta):
    J, H = oracle_mod.m1_JH(V[0], V[1:], v, W, gl, gu, dthin, dthick)
    vl = gl @ v
    Sn = W * ((eta + ks * J) - (ka + ks) * (V[0] - V[1:] @ v))
    Si = W * (eta - ka * J) * vl - (ka + ks) * H
    return alpha * np.concatenate([[Sn], Si])


def test_jacobian_matches_finite_differences(oracle_mod):
    rng = np.random.default_rng(4)
    for _ in range(10):
        E, F, v, W, gl, gu = _rand_state(rng)
        dthick = rng.uniform(0.0, 1.0)
        dthin = 1.0 - dthick
        alpha, ka, ks, eta = 0.8, 0.7, 0.4, 0.0          # the Jacobian does not depend on eta; eta >> E would only add rounding noise to the differences
        Jac = oracle_mod.m1_jacobian(E, F, v, W, gl, gu, dthin, dthick, alpha, ka, ks)
        V = np.concatenate([[E], F])
        for j in range(4):
            h = 1e-6 * E
            Vp, Vm = V.copy(), V.copy()
            Vp[j] += h
            Vm[j] -= h
            fd = (_RV(oracle_mod, Vp, v, W, gl, gu, dthin, dthick, alpha, ka, ks, eta) -
                  _RV(oracle_mod, Vm, v, W, gl, gu, dthin, dthick, alpha, ka, ks, eta)) / (2 * h)
            assert np.abs(fd - Jac[:, j]).max() < 1e-7 * np.abs(Jac).max(), (j, fd, Jac[:, j])


def _oracle(oracle_mod, **over):
    return oracle_mod.Oracle(synth.default_params(**over), 4, 4, 4, 3, 0.1)


def test_implicit_solve_limits(oracle_mod):
    rng = np.random.default_rng(5)
    E, F, v, W, gl, gu = _rand_state(rng, vmax=0.3)
    Vs = np.concatenate([[1e-4, E], F])
    # no interaction: V = V*
    o = _oracle(oracle_mod, m1_kappa0=0.0)
    V, R, fl = o.m1_implicit_point(0, Vs, 0.1, 0.9, v, W, 1e-3, 0.02, gl, gu)
    assert fl == 0 and np.array_equal(V, Vs) and np.all(R == 0.0)
    # residual of (C13)-(C14) and (C10) at return
    o = _oracle(oracle_mod, m1_kappa0=5.0)
    for adt in (1e-3, 0.1, 10.0):
        V, R, fl = o.m1_implicit_point(0, Vs, adt, 0.9, v, W, 1e-3, 0.3, gl, gu)
        assert fl == 0
        assert np.abs(V - Vs - adt * R).max() < 1e-12 * max(E, np.abs(V).max())
    # v = 0, kappa dt -> infinity: J -> eta / kappa_a, H -> 0 (thermal equilibrium)
    o = _oracle(oracle_mod, m1_kappa0=1e9)
    V, R, fl = o.m1_implicit_point(0, Vs, 1.0, 1.0, np.zeros(3), 1.0, 1e-3, 0.3, ID, ID)
    assert abs(V[1] / 0.3 ** 4 - 1) < 1e-8 and np.abs(V[2:]).max() < 1e-8 * V[1]
    # v = 0: the system is linear; compare with the direct solve of Eq. (C6)
    ka = 5.0 * 1.0
    o = _oracle(oracle_mod, m1_kappa0=5.0)
    al, adt, T = 0.9, 0.2, 0.3
    V, R, fl = o.m1_implicit_point(0, Vs, adt, al, np.zeros(3), 1.0, 1e-3, T, ID, ID)
    Eex = (Vs[1] + adt * al * ka * T ** 4) / (1 + adt * al * ka)          # S_n = eta - kappa_a E  (J = E at v = 0)
    Fex = Vs[2:] / (1 + adt * al * 2 * ka)                                # S_i = -(kappa_a + kappa_s) F_i
    assert abs(V[1] / Eex - 1) < 1e-12 and np.abs(V[2:] - Fex).max() < 1e-12 * np.abs(Fex).max()
    Nex = (Vs[0] + adt * al * ka * T ** 4) / (1 + adt * al * ka)          # Gamma = 1
    assert abs(V[0] / Nex - 1) < 1e-12


def test_m1_rhs_constant_state_and_diffusion_limit(oracle_mod):
    """Flat space, uniform fluid at rest, uniform radiation: flux divergence and geometric sources vanish exactly;
    optically thick limit of Eq. (77): A -> 0 gives the centred flux (F_i + F_i+1)/2."""
    n, ng, dx = 8, 3, 0.1
    o = oracle_mod.Oracle(synth.default_params(), n, n, n, ng, dx)
    U = synth._flat_state(o.shape)
    P = np.zeros((10,) + o.shape)
    P[synth.RHO], P[synth.WLOR], P[synth.TEMP] = 1e-3, 1.0, 0.01
    V = np.zeros((15,) + o.shape)
    for s in range(3):
        V[5 * s], V[5 * s + 1], V[5 * s + 2] = 1e-4, 1e-5, 2e-6
    KV = o.m1_rhs(U, P, V)
    assert np.all(KV == 0.0)
    # smooth E profile, F = 0, huge opacity: dF_x/dt = -d_x (E/3) with the centred 2nd-order difference
    o2 = oracle_mod.Oracle(synth.default_params(m1_kappa0=1e12), n, n, n, ng, dx)
    X = synth.mesh(n, n, n, ng, dx)[0]
    V[:] = 0.0
    V[1] = 1e-5 * (1.0 + 0.1 * np.sin(2 * math.pi * X / (n * dx)))
    V[6] = V[11] = 1e-5
    KV = o2.m1_rhs(U, P, V)
    I = (slice(ng, -ng),) * 3
    ref = -(V[1][:, :, ng + 1:-ng + 1 or None] - V[1][:, :, ng - 1:-ng - 1]) / (2 * dx) / 3.0
    assert np.abs(KV[2][I] - ref[ng:-ng, ng:-ng]).max() < 1e-12 * np.abs(ref).max()


def test_imex_tableau_conditions():
    """R1: the conditions PAPER.md:389-410 states for IMEX(3,3,2): the explicit half is the Shu-Osher SSP-RK(3,3) (its weights are
    Eq. 59 at theta = 1), the implicit half is a DIRK with c_i = sum_j a_ij (Eq. 55), second order incl. the mixed conditions,
    L-stable. Catches: a non-SSP explicit half (the round-1 tableau), a wrong sign in a_21, a diagonal that is not L-stable."""
    ae, we, ai, wi = synth.imex_tableau()
    a3, w3 = synth.tableau("ssprk3")
    assert np.array_equal(ae, a3) and np.array_equal(we, w3)
    assert np.allclose(ae.sum(axis=1), [0.0, 1.0, 0.5])
    b = lambda th: np.array([th - 5.0 / 6.0 * th * th, th * th / 6.0, 4.0 * th * th / 6.0])      # Eq. (59)
    assert np.allclose(b(1.0), we, atol=1e-15)
    # explicit half: third order
    ce, ci = ae.sum(axis=1), ai.sum(axis=1)
    assert abs(we @ ce ** 2 - 1 / 3) < 1e-15 and abs(we @ (ae @ ce) - 1 / 6) < 1e-15
    assert np.allclose(np.triu(ae), 0) and np.allclose(np.triu(ai, 1), 0)
    assert abs(we.sum() - 1) < 1e-15 and abs(wi.sum() - 1) < 1e-15
    for w in (we, wi):
        for c in (ce, ci):
            assert abs(w @ c - 0.5) < 1e-15
    assert abs(1.0 - wi @ np.linalg.solve(ai, np.ones(3))) < 1e-14      # R(-inf) = 0: L-stable
    # A-stability on the imaginary axis: |R(iy)| <= 1
    for y in np.linspace(0.0, 50.0, 201):
        z = 1j * y
        R = 1.0 + z * (wi @ np.linalg.solve(np.eye(3) - z * ai, np.ones(3)))
        assert abs(R) <= 1.0 + 1e-12


def test_odd_even_switch_fires_on_a_zigzag_only(oracle_mod):
    """l.565-570 with reading R33: on a genuine zigzag (alternating E) in an optically thick medium the switch sets A = 1 and the
    full Lax-Friedrichs dissipation acts; with the switch off the same data see A = tanh(1/(kappa dx)) ~ 0; on a smooth profile
    with rounding-level noise the switch must NOT fire."""
    n, ng, dx = 12, 3, 0.1
    U = synth._flat_state((n + 6,) * 3)
    P = np.zeros((10,) + U.shape[1:])
    P[synth.RHO], P[synth.WLOR], P[synth.TEMP] = 1e-3, 1.0, 0.01
    idx = np.arange(n + 6)
    zig = 1e-5 * (1.0 + 0.1 * (-1.0) ** idx)[None, None, :] * np.ones(U.shape[1:])
    V = np.zeros((15,) + U.shape[1:])
    V[1] = zig
    V[6] = V[11] = 1e-5
    I = (slice(ng, -ng),) * 3
    out = {}
    for oe in (0, 1):
        o = oracle_mod.Oracle(synth.default_params(m1_kappa0=1e6, m1_odd_even=oe), n, n, n, ng, dx)
        out[oe] = o.m1_rhs(U, P, V)[1][I]
    # switch off: A ~ 1e-5, the E equation sees (almost) no dissipation; switch on: -lambda (u_{i+1} - 2 u_i + u_{i-1}) / (2 dx) with lambda = 1/sqrt3
    assert np.abs(out[0]).max() < 1e-3 * np.abs(out[1]).max()
    lap = (zig[:, :, ng + 1:n + ng + 1] - 2 * zig[:, :, ng:n + ng] + zig[:, :, ng - 1:n + ng - 1])[ng:-ng, ng:-ng]
    lam = 1.0 / np.sqrt(3.0)                       # (B5) thick limit at rest: sqrt(3 gamma^xx) / 3
    assert np.abs(out[1] - 0.5 * lam * lap / dx).max() < 1e-9 * np.abs(out[1]).max()
    # smooth profile + rounding noise: both settings agree
    rng = np.random.default_rng(0)
    X = synth.mesh(n, n, n, ng, dx)[0]
    V[1] = 1e-5 * (1.0 + 0.1 * np.sin(2 * np.pi * X / (n * dx))) * (1.0 + 1e-15 * rng.standard_normal(X.shape))
    res = []
    for oe in (0, 1):
        o = oracle_mod.Oracle(synth.default_params(m1_kappa0=1e6, m1_odd_even=oe), n, n, n, ng, dx)
        res.append(o.m1_rhs(U, P, V)[1][I])
    assert np.array_equal(res[0], res[1])


def test_radiation_gravitates_like_an_equal_fluid(oracle_mod):
    """R6, second half: radiation that is isotropic in the frame of a fluid moving with v^i (H = 0: the closure is exact there)
    has the stress-energy of a perfect fluid with p = e / 3 moving with the same v^i. The matter sources of Eqs. (14), (16),
    (17), (19) are linear in T^ab, so  rhs(fluid A + radiation) - rhs(fluid A) = rhs(fluid R) - rhs(vacuum)  to rounding, with
    fluid R: Gamma - 1 = (1 + eps_R) / (3 eps_R). Spacetime: the perturbed one of config 1 (non-trivial alpha, chi, gamma~_ij)."""
    cfg = synth.config1(n=8, gauge_perturbation=True)
    n = cfg["n"]
    vu = (0.2, -0.1, 0.15)

    def spacetime_rhs(rho, eps, gamma, moving, V=None, grav_G=1.0):
        par = synth.default_params(eos_gamma=gamma, grav_G=grav_G)
        o = oracle_mod.Oracle(par, n[0], n[1], n[2], cfg["ng"], cfg["dx"])
        U, P = cfg["U"].copy(), np.zeros_like(cfg["P"])
        U[28:32] = 0.0                                   # no magnetic field, no cleaning scalar
        P[synth.RHO], P[synth.EPS], P[synth.YE] = rho, eps, 0.3
        for i in range(3):
            P[synth.VX + i] = vu[i] if moving else 0.0
        o.prim2con(U, P)
        Pc, F = o.con2prim(U)
        K = o.rhs(U, Pc, "ccz4")
        if V is not None:
            o.m1_gravity(U, Pc, V, K)
        return K[:22, 3:-3, 3:-3, 3:-3], U, Pc

    X = synth.mesh(n[0], n[1], n[2], cfg["ng"], cfg["dx"])[0]
    J = 4e-4 * (1.0 + 0.2 * np.sin(2 * np.pi * X / (n[0] * cfg["dx"])))      # comoving energy density of the radiation
    KA, U, Pc = spacetime_rhs(1e-3, 0.1, 2.0, True)
    chi = U[synth.CHI]
    gl = [[U[synth.SYM[i][j]] / chi for j in range(3)] for i in range(3)]
    vl = [sum(gl[i][j] * vu[j] for j in range(3)) for i in range(3)]
    W2 = 1.0 / (1.0 - sum(vl[i] * vu[i] for i in range(3)))
    assert np.abs(Pc[synth.WLOR] ** 2 / W2 - 1).max() < 1e-12
    E = 4.0 / 3.0 * J * W2 - J / 3.0
    sg = chi ** -1.5
    V = np.zeros((15,) + X.shape)
    for s, w in enumerate((0.5, 0.3, 0.2)):              # split over the three species
        V[5 * s] = 1e-30
        V[5 * s + 1] = sg * w * E
        for i in range(3):
            V[5 * s + 2 + i] = sg * w * 4.0 / 3.0 * J * W2 * vl[i]
    KAR, _, _ = spacetime_rhs(1e-3, 0.1, 2.0, True, V)
    eps_R = 500.0                                        # below eps_max = 1e3 of the error policy
    KR, _, _ = spacetime_rhs(J / (1.0 + eps_R), eps_R, 1.0 + (1.0 + eps_R) / (3.0 * eps_R), True)
    K0, _, _ = spacetime_rhs(1e-3, 0.1, 2.0, False, grav_G=0.0)   # geometry alone: matter decoupled (R29)
    lhs, rhs_ = KAR - KA, KR - K0
    scale = np.abs(rhs_).reshape(22, -1).max(axis=1)
    live = scale > 1e-12
    assert live.sum() >= 11                              # K^, Theta, six A~_ij, three Gamma^^i
    err = np.abs(lhs - rhs_).reshape(22, -1).max(axis=1)
    assert np.all(err[live] < 1e-8 * scale[live]), (err / np.maximum(scale, 1e-300), scale)
    assert np.all(err[~live] < 1e-14)


def test_static_radial_beam_in_schwarzschild(oracle_mod):
    """Pin of the flux brackets AND the geometric sources of Eqs. (38)-(40) in a curved, static spacetime: radiation streaming
    radially outwards in the Schwarzschild metric in isotropic coordinates (alpha = (1 - M/2r)/(1 + M/2r), gamma_ij = psi^4 delta_ij,
    psi = 1 + M/2r) is stationary when  alpha^2 psi^6 r^2 F^r = const  (d_r (sqrt(-g) T^r_t) = 0),  E = |F| = psi^2 F^r (free
    streaming) and N = alpha E (number flux alpha psi^6 r^2 N F^r / E = const; E = N x local energy ~ N / alpha): energy redshifts,
    number does not.
    The explicit part F_V of the oracle must then vanish at the order of its centred fluxes (second)."""
    M, C = 1.0, 1e-3
    res = {}
    for n in (16, 32):
        ng, L = 3, 4.0
        dx = L / n
        o = oracle_mod.Oracle(synth.default_params(m1_kappa0=0.0), n, n, n, ng, dx)
        X, Y, Z = synth.mesh(n, n, n, ng, dx, x0=(4.0, -2.0, -2.0))
        r = np.sqrt(X * X + Y * Y + Z * Z)
        psi = 1.0 + M / (2 * r)
        alpha = (1.0 - M / (2 * r)) / psi
        U = synth._flat_state(X.shape)
        U[synth.CHI], U[synth.ALPHA] = psi ** -4, alpha
        P = np.zeros((10,) + X.shape)
        P[synth.RHO], P[synth.WLOR], P[synth.TEMP] = 1e-10, 1.0, 1e-8
        Fr = C / (alpha ** 2 * psi ** 6 * r * r)              # F^r
        E = psi ** 2 * Fr
        sg = psi ** 6
        V = np.zeros((15,) + X.shape)
        for s in range(3):
            V[5 * s] = sg * E * alpha
            V[5 * s + 1] = sg * E
            for i, xi in enumerate((X, Y, Z)):
                V[5 * s + 2 + i] = sg * psi ** 4 * Fr * xi / r    # F_i = gamma_ij F^j
        KV = o.m1_rhs(U, P, V)
        I = (slice(ng, -ng),) * 3
        # scale of the individual terms that must cancel: alpha F^x sqrt(gamma) / r ~ flux / length
        scaleE = np.abs(alpha * sg * Fr / r)[I].max()
        res[n] = [np.abs(KV[f][I]).max() / scaleE for f in range(5)]
    for f in range(5):
        assert res[32][f] < 0.02, res                          # O(dx^2) of the cancelling terms (dx = 0.125, gradients ~ 1/r)
        assert res[16][f] / res[32][f] > 3.0, (f, res)         # second-order convergence to the stationary state
