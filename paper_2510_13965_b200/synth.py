"""Seeded synthetic inputs for the MHDuet patch hot path (numpy only).

This module serves BOTH the oracle (tests) and the CUDA library (tests, bench, smoke). It holds
none of the method's arithmetic: it produces *initial data* — spacetime fields in the conformal
variables of PAPER.md:132, primitive fluid fields (rho, Ye, eps, v^i), the densitised magnetic
field and the parameter dictionaries / Butcher tableaux. The conserved fluid fields are produced
from these by `prim2con` of whichever implementation is under test.

The recipes stand in for the paper's neutron-star workloads (Sec. V), whose EoS tables, opacity
tables and initial data are not available; see DESIGN.md "Input recipe".

State layout (32 fields, SoA, array shape (32, MZ, MY, MX), x fastest):
  0-5 gamma~_ij (xx,xy,xz,yy,yz,zz)  6-11 A~_ij  12 chi  13 K^  14 Theta  15-17 Gamma^^i
  18 alpha  19-21 beta^i  22 Dbar  23 DYebar  24 taubar  25-27 Sbar_i  28-30 Bbar^i  31 phibar
Primitive layout (10 fields): rho, Ye, eps, p, v^x, v^y, v^z, W, T, cs2.
"""
import math

import numpy as np

NSTATE, NPRIM, NG = 32, 10, 3
GXX, AXX, CHI, KHAT, THETA, GAMX, ALPHA, BETAX = 0, 6, 12, 13, 14, 15, 18, 19
DBAR, DYEBAR, TAUBAR, SXBAR, BXBAR, PHIBAR = 22, 23, 24, 25, 28, 31
RHO, YE, EPS, PRESS, VX, WLOR, TEMP, CS2 = 0, 1, 2, 3, 4, 7, 8, 9
SYM = ((0, 1, 2), (1, 3, 4), (2, 4, 5))
SEED_BASE = 2510139650
_MASK = (1 << 64) - 1


class SplitMix64:
    """Counter-based 64-bit generator; uniform(a,b) = a + (b-a) * (next()>>11) * 2^-53."""

    def __init__(self, seed):
        self.s = seed & _MASK

    def next(self):
        self.s = (self.s + 0x9E3779B97F4A7C15) & _MASK
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
        return z ^ (z >> 31)

    def uniform(self, a=0.0, b=1.0):
        return a + (b - a) * ((self.next() >> 11) * 2.0 ** -53)

    def randint(self, lo, hi):
        """integer in [lo, hi]"""
        return lo + self.next() % (hi - lo + 1)


# ---- Butcher tableaux (R2): caller data for mhd_rk_stage / Oracle.evolve -------------------------
def tableau(name):
    """Explicit tableaux named in PAPER.md:400 (textbook forms; weights equal Eqs. 58-59 at theta=1)."""
    if name == "rk4":
        a = np.zeros((4, 4))
        a[1, 0] = 0.5
        a[2, 1] = 0.5
        a[3, 2] = 1.0
        w = np.array([1 / 6, 1 / 3, 1 / 3, 1 / 6])
    elif name == "ssprk3":
        a = np.zeros((3, 3))
        a[1, 0] = 1.0
        a[2, 0] = 0.25
        a[2, 1] = 0.25
        w = np.array([1 / 6, 1 / 6, 2 / 3])
    else:
        raise ValueError(name)
    return a, w


def imex_tableau(name="imex332"):
    """IMEX pair (a_expl, w_expl, a_impl, w_impl) in the form of PAPER.md Eqs. (53)-(55) for IMEX(3,3,2) (l.408-410): the explicit
    half IS the Shu-Osher SSP-RK(3,3) the paper names (tableau('ssprk3')). The body of the paper's Table II (I32L(3,2)) is
    missing (R1), so the implicit half is caller data; the default is the 3-stage, 2nd-order, L-stable DIRK with constant
    diagonal g = 1 - 1/sqrt(2) and the same weights as the explicit half (the published IMEX-SSP3(3,3,2) pairing): it meets
    every condition the paper states (sum w = 1, sum w c = sum w c~ = sum w~ c = sum w~ c~ = 1/2, DIRK, c_i = sum_j a_ij,
    R(-inf) = 0); `tests/test_oracle_m1.py::test_imex_tableau_conditions` checks them."""
    if name != "imex332":
        raise ValueError(name)
    ae, we = tableau("ssprk3")
    g = 1.0 - 1.0 / math.sqrt(2.0)
    ai = np.zeros((3, 3))
    ai[0, 0] = ai[1, 1] = ai[2, 2] = g
    ai[1, 0] = 1.0 - 2.0 * g
    ai[2, 0] = 0.5 - g
    wi = we.copy()
    return ae, we, ai, wi


# ---- parameters ------------------------------------------------------------------------------------
def default_params(**over):
    """Parameter dictionary (R3, R10, R16, R18 defaults; all damping terms non-zero so they are exercised)."""
    p = dict(
        eos_kind=0, eos_gamma=2.0, eos_gamma_th=2.0, n_pieces=1,
        pp_K=[100.0], pp_Gamma=[2.0], pp_rho=[1e300],
        kappa_z=0.5, kappa_c=0.05, kappa_2=0.0, eta_shift=1.0, f_alpha=1.0, f_beta=1.0, beta0=[0.0, 0.0, 0.0],
        grav_G=1.0, sigma_ko_spacetime=0.1, sigma_ko_matter=0.0,
        c_b=1.0, kappa_b=1.0, mp5_alpha=4.0,
        rho_atmo=1e-10, rho_cut=1.01e-10, rho_low=1e-8, alpha_bh=0.1, w_max=100.0, rho_max=1.0,
        eps_min=0.0, eps_max=1e3, ye_min=0.0, ye_max=1.0, ye_atmo=0.3, eps_atmo=1e-8, T_atmo=0.1,
        c2p_maxit=100,
        m1_kappa0=1e-6, m1_rho0=1e-3, m1_species_scale=[1.0, 0.8, 0.5], m1_efloor=1e-30, m1_tol=1e-13, m1_mb=1.0, m1_maxit=30, m1_odd_even=1, m1_arad=1.0, m1_oe_guard=1e-10,
        recon_kind=0, weno_eps=1e-6, les_C_M=0.0, les_C_N=0.0, les_C_Y=0.0, les_C_T=0.0,
    )
    p.update(over)
    return p


# ---- grid helpers ----------------------------------------------------------------------------------
def coords(n, ng, dx, x0=0.0):
    """vertex-centred coordinates incl. ghosts: x_i = x0 + (i - ng) dx"""
    return x0 + (np.arange(n + 2 * ng) - ng) * dx


def mesh(nx, ny, nz, ng, dx, x0=(0.0, 0.0, 0.0)):
    x = coords(nx, ng, dx, x0[0])
    y = coords(ny, ng, dx, x0[1])
    z = coords(nz, ng, dx, x0[2])
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    return X, Y, Z


def _inv3(g):
    """inverse and determinant of symmetric 3x3 fields g[i][j] (arrays)"""
    det = (g[0][0] * (g[1][1] * g[2][2] - g[1][2] * g[1][2]) - g[0][1] * (g[0][1] * g[2][2] - g[1][2] * g[0][2])
           + g[0][2] * (g[0][1] * g[1][2] - g[1][1] * g[0][2]))
    gi = [[None] * 3 for _ in range(3)]
    gi[0][0] = (g[1][1] * g[2][2] - g[1][2] * g[1][2]) / det
    gi[0][1] = gi[1][0] = (g[0][2] * g[1][2] - g[0][1] * g[2][2]) / det
    gi[0][2] = gi[2][0] = (g[0][1] * g[1][2] - g[0][2] * g[1][1]) / det
    gi[1][1] = (g[0][0] * g[2][2] - g[0][2] * g[0][2]) / det
    gi[1][2] = gi[2][1] = (g[0][1] * g[0][2] - g[0][0] * g[1][2]) / det
    gi[2][2] = (g[0][0] * g[1][1] - g[0][1] * g[0][1]) / det
    return gi, det


def conformal_from_adm(gam, dgam, Kij, alpha, beta, theta=None, Zup=None):
    """Initial-data bookkeeping: physical (gamma_ij, d_k gamma_ij, K_ij) -> the 22 conformal fields of
    PAPER.md:132 with Gamma^^i = Gamma~^i (+ 2 Z^i / chi) from the analytic derivatives.
    gam[i][j], Kij[i][j]: arrays; dgam[k][i][j]: arrays; beta[i]; returns array (22, ...)."""
    shape = np.shape(alpha)
    gi, det = _inv3(gam)
    chi = det ** (-1.0 / 3.0)
    # d_k chi = -(1/3) chi gamma^ij d_k gamma_ij
    dchi = [-(chi / 3.0) * sum(gi[i][j] * dgam[k][i][j] for i in range(3) for j in range(3)) for k in range(3)]
    gt = [[chi * gam[i][j] for j in range(3)] for i in range(3)]
    dgt = [[[dchi[k] * gam[i][j] + chi * dgam[k][i][j] for j in range(3)] for i in range(3)] for k in range(3)]
    gti, _ = _inv3(gt)
    trK = sum(gi[i][j] * Kij[i][j] for i in range(3) for j in range(3))
    out = np.zeros((22,) + shape)
    for i in range(3):
        for j in range(i, 3):
            out[GXX + SYM[i][j]] = gt[i][j]
            out[AXX + SYM[i][j]] = chi * (Kij[i][j] - gam[i][j] * trK / 3.0)
    th = 0.0 if theta is None else theta
    out[CHI] = chi
    out[THETA] = th
    out[KHAT] = trK - 2.0 * th
    for k in range(3):
        # Gamma~^k = gamma~^ij gamma~^kl (d_i gamma~_lj - 1/2 d_l gamma~_ij)
        G = sum(gti[i][j] * gti[k][l] * (dgt[i][l][j] - 0.5 * dgt[l][i][j])
                for i in range(3) for j in range(3) for l in range(3))
        out[GAMX + k] = G + (0.0 if Zup is None else 2.0 * Zup[k] / chi)
    out[ALPHA] = alpha
    for k in range(3):
        out[BETAX + k] = beta[k]
    return out


# ---- config 1: perturbed flat spacetime + smooth magnetised ideal gas (BASELINE.json configs[0]) ----
def config1(n=32, dx=0.1, seed=SEED_BASE + 1, gauge_perturbation=False, ng=NG):
    """Periodic box of n^3 interior points. gamma_ij = delta_ij + sum_m A^m_ij sin(k^m.x + phi^m),
    K_ij = -1/2 d_t h_ij for waves h(k.x - |k| t), alpha=1, beta=0 (or perturbed if gauge_perturbation,
    which also seeds Theta and a Gamma^ offset so that every CCZ4 term is exercised).
    Draw order: 3 metric modes x (n_x,n_y,n_z, phase, 6 amplitudes); 3 density modes; 3 modes per velocity
    component; vector-potential mode; Ye mode; [gauge modes]."""
    rng = SplitMix64(seed)
    L = n * dx
    X, Y, Z = mesh(n, n, n, ng, dx)
    k0 = 2.0 * math.pi / L

    def mode():
        kv = [k0 * rng.randint(1, 3) for _ in range(3)]
        ph = rng.uniform(0.0, 2.0 * math.pi)
        return kv, ph

    def phase(kv, ph):
        return kv[0] * X + kv[1] * Y + kv[2] * Z + ph

    one = np.ones_like(X)
    gam = [[one * (1.0 if i == j else 0.0) for j in range(3)] for i in range(3)]
    dgam = [[[np.zeros_like(X) for _ in range(3)] for _ in range(3)] for _ in range(3)]
    Kij = [[np.zeros_like(X) for _ in range(3)] for _ in range(3)]
    for _ in range(3):
        kv, ph = mode()
        om = math.sqrt(sum(c * c for c in kv))
        th = phase(kv, ph)
        s, c = np.sin(th), np.cos(th)
        for (i, j) in ((0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)):
            A = rng.uniform(-1e-4, 1e-4)
            for (a, b) in {(i, j), (j, i)}:
                gam[a][b] = gam[a][b] + A * s
                Kij[a][b] = Kij[a][b] + 0.5 * om * A * c
                for k in range(3):
                    dgam[k][a][b] = dgam[k][a][b] + A * kv[k] * c
    rho = 1.0e-3 * one
    for _ in range(3):
        kv, ph = mode()
        rho = rho + 1.0e-3 * (0.1 / 3.0) * np.sin(phase(kv, ph))
    v = []
    for _ in range(3):
        vi = np.zeros_like(X)
        for _ in range(3):
            kv, ph = mode()
            vi = vi + (rng.uniform(-0.1, 0.1) / 3.0) * np.sin(phase(kv, ph))
        v.append(vi)
    kv, ph = mode()
    avec = [rng.uniform(-1e-4, 1e-4) for _ in range(3)]
    cth = np.cos(phase(kv, ph))
    B = [(kv[1] * avec[2] - kv[2] * avec[1]) * cth, (kv[2] * avec[0] - kv[0] * avec[2]) * cth,
         1.0e-3 + (kv[0] * avec[1] - kv[1] * avec[0]) * cth]
    kv, ph = mode()
    ye = 0.3 + 0.05 * np.sin(phase(kv, ph))
    alpha, beta, theta, Zup = one.copy(), [np.zeros_like(X) for _ in range(3)], None, None
    if gauge_perturbation:
        kv, ph = mode()
        alpha = 1.0 + 0.05 * np.sin(phase(kv, ph))
        for i in range(3):
            kv, ph = mode()
            beta[i] = 0.03 * np.sin(phase(kv, ph))     # both signs -> both upwind branches
        kv, ph = mode()
        theta = 1e-3 * np.sin(phase(kv, ph))
        Zup = []
        for i in range(3):
            kv, ph = mode()
            Zup.append(1e-3 * np.cos(phase(kv, ph)))
    U = np.zeros((NSTATE,) + X.shape)
    U[:22] = conformal_from_adm(gam, dgam, Kij, alpha, beta, theta, Zup)
    sg = U[CHI] ** -1.5
    for i in range(3):
        U[BXBAR + i] = sg * B[i]
    if gauge_perturbation:
        kv, ph = mode()
        U[PHIBAR] = sg * 1e-5 * np.sin(phase(kv, ph))
    P = np.zeros((NPRIM,) + X.shape)
    P[RHO], P[YE], P[EPS] = rho, ye, 0.1
    for i in range(3):
        P[VX + i] = v[i]
    return dict(U=U, P=P, n=(n, n, n), ng=ng, dx=dx, bc=[0] * 6, params=default_params())


# ---- flat-space helpers -------------------------------------------------------------------------------
def _flat_state(shape):
    """22 spacetime fields of Minkowski space in the conformal variables: gamma~ = delta, chi = 1, alpha = 1, rest 0."""
    U = np.zeros((NSTATE,) + shape)
    U[GXX + 0] = U[GXX + 3] = U[GXX + 5] = 1.0
    U[CHI] = 1.0
    U[ALPHA] = 1.0
    return U


# ---- config 2: smooth convergence series (BASELINE.json configs[1]) ---------------------------------------
def config2_gauge_wave(n=32, amplitude=1e-6, t=0.0, ng=NG, ny=None):
    """Linearised gauge wave, 1-D in 3-D along x on the unit box: alpha = 1 + A sin k(x - sqrt2 t),
    K = (sqrt2/2) A k cos k(x - sqrt2 t), flat metric, zero shift (f_beta = eta = 0), vacuum-like fluid (atmosphere,
    grav_G = 0). Solves the linearised Eqs. (16), (25) (1+log slicing: speed sqrt 2); error floor O(A^2).
    Returns the same dict as config1 plus `exact(t)` -> (alpha, Khat) arrays."""
    L = 1.0
    dx = L / n
    ny = n if ny is None else ny                 # ny < n: thin slab for the (cheap) 1-D convergence pins
    X, Y, Z = mesh(n, ny, ny, ng, dx)
    k = 2.0 * math.pi / L

    def exact(tt):
        ph = k * (X - math.sqrt(2.0) * tt)
        return 1.0 + amplitude * np.sin(ph), 0.5 * math.sqrt(2.0) * amplitude * k * np.cos(ph)

    U = _flat_state(X.shape)
    U[ALPHA], U[KHAT] = exact(t)
    P = np.zeros((NPRIM,) + X.shape)
    par = default_params(f_beta=0.0, eta_shift=0.0, kappa_z=0.0, kappa_c=0.0, grav_G=0.0)
    P[RHO], P[YE], P[EPS] = par["rho_atmo"], par["ye_atmo"], par["eps_atmo"]
    return dict(U=U, P=P, n=(n, ny, ny), ng=ng, dx=dx, bc=[0] * 6, params=par, exact=exact, L=L)


def config2_alfven(n=32, t=0.0, ng=NG, rho=1.0, p=1.0, B0=1.0, eta=1.0, gamma=5.0 / 3.0, ny=None):
    """Circularly polarised Alfven wave of arbitrary amplitude (an exact SRMHD solution; ref. [99] of the paper),
    1-D in 3-D along x on the unit box, flat spacetime with grav_G = 0 so that the metric stays exactly flat.
    B^x = B0, B^y = eta B0 cos k(x - vA t), B^z = eta B0 sin k(x - vA t), v^x = 0, v^{y,z} = -vA B^{y,z} / B0."""
    L = 1.0
    dx = L / n
    ny = n if ny is None else ny                 # ny < n: thin slab for the (cheap) 1-D convergence pins
    X, Y, Z = mesh(n, ny, ny, ng, dx)
    k = 2.0 * math.pi / L
    eps = p / ((gamma - 1.0) * rho)
    rhoh = rho * (1.0 + eps) + p
    den = rhoh + B0 * B0 * (1.0 + eta * eta)
    vA = math.sqrt(B0 * B0 / den / (0.5 * (1.0 + math.sqrt(1.0 - (2.0 * eta * B0 * B0 / den) ** 2))))

    def exact(tt):
        ph = k * (X - vA * tt)
        By, Bz = eta * B0 * np.cos(ph), eta * B0 * np.sin(ph)
        return dict(B=[np.full_like(X, B0), By, Bz], v=[np.zeros_like(X), -vA * By / B0, -vA * Bz / B0])

    U = _flat_state(X.shape)
    e0 = exact(t)
    P = np.zeros((NPRIM,) + X.shape)
    P[RHO], P[YE], P[EPS] = rho, 0.3, eps
    for i in range(3):
        U[BXBAR + i] = e0["B"][i]
        P[VX + i] = e0["v"][i]
    par = default_params(eos_gamma=gamma, grav_G=0.0, rho_max=1e3, kappa_z=0.0, kappa_c=0.0)
    return dict(U=U, P=P, n=(n, ny, ny), ng=ng, dx=dx, bc=[0] * 6, params=par, exact=exact, L=L, vA=vA)


def riemann_1d(n=128, ng=NG, ny=4):
    """1-D magnetised Riemann problem (Balsara-1 type states) along x on [-0.5, 0.5], outflow in x, periodic in y, z;
    flat spacetime with grav_G = 0. Used for the monotonicity pin of the flux-splitting MP5 scheme."""
    dx = 1.0 / n
    X, Y, Z = mesh(n, ny, ny, ng, dx, x0=(-0.5 + 0.5 * dx, 0.0, 0.0))
    left = X < 0.0
    gamma = 2.0
    U = _flat_state(X.shape)
    P = np.zeros((NPRIM,) + X.shape)
    P[RHO] = np.where(left, 1.0, 0.125)
    pr = np.where(left, 1.0, 0.1)
    P[EPS] = pr / ((gamma - 1.0) * P[RHO])
    P[YE] = 0.3
    U[BXBAR], U[BXBAR + 1] = 0.5, np.where(left, 1.0, -1.0)
    par = default_params(eos_gamma=gamma, grav_G=0.0, rho_max=1e3, kappa_z=0.0, kappa_c=0.0)
    return dict(U=U, P=P, n=(n, ny, ny), ng=ng, dx=dx, bc=[1, 1, 0, 0, 0, 0], params=par)


# ---- TOV star in isotropic coordinates (initial data for configs 3-5) ---------------------------------------
_TOV_CACHE = {}


def tov_profile(K, Gamma, rho_c, dr=2.0e-3):
    """Textbook TOV equations in the areal radius r for the polytrope p = K rho^Gamma, eps = p / ((Gamma-1) rho),
    integrated with classical RK4 from the centre to the surface, together with the map to the isotropic radius rbar:
      dm/dr = 4 pi r^2 e,  dp/dr = -(e + p)(m + 4 pi r^3 p) / (r (r - 2m)),  dnu/dr = (m + 4 pi r^3 p) / (r (r - 2m)),
      d ln(rbar/r)/dr = (1/sqrt(1 - 2m/r) - 1) / r,   e = rho (1 + eps),
    normalised to the exterior solution rbar = (r - M + sqrt(r^2 - 2 M r)) / 2, alpha = (1 - M/2rbar)/(1 + M/2rbar).
    Returns a dict of 1-D arrays over rbar (interior) and the scalars M, Rbar."""
    key = (K, Gamma, rho_c, dr)
    if key in _TOV_CACHE:
        return _TOV_CACHE[key]

    def eos(p):
        rho = (max(p, 0.0) / K) ** (1.0 / Gamma)
        return rho, rho + max(p, 0.0) / (Gamma - 1.0)

    def rhs(r, y):
        m, p, nu, lq = y
        rho, e = eos(p)
        if r == 0.0:
            return np.array([0.0, 0.0, 0.0, 0.0])
        a = (m + 4.0 * math.pi * r ** 3 * p) / (r * (r - 2.0 * m))
        return np.array([4.0 * math.pi * r * r * e, -(e + p) * a, a, (1.0 / math.sqrt(1.0 - 2.0 * m / r) - 1.0) / r])

    p_c = K * rho_c ** Gamma
    y = np.array([0.0, p_c, 0.0, 0.0])
    r = 0.0
    rs, ys = [r], [y.copy()]
    p_stop = 1e-12 * p_c
    while y[1] > p_stop and r < 100.0:
        k1 = rhs(r, y)
        k2 = rhs(r + 0.5 * dr, y + 0.5 * dr * k1)
        k3 = rhs(r + 0.5 * dr, y + 0.5 * dr * k2)
        k4 = rhs(r + dr, y + dr * k3)
        yn = y + dr / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
        if yn[1] <= p_stop:                      # last partial step to the surface by linear interpolation in p
            f = (y[1] - p_stop) / (y[1] - yn[1])
            yn = y + f * (yn - y)
            r += f * dr
            yn[1] = 0.0
            rs.append(r)
            ys.append(yn)
            break
        r += dr
        y = yn
        rs.append(r)
        ys.append(y.copy())
    rs, ys = np.array(rs), np.array(ys)
    M, R = ys[-1, 0], rs[-1]
    Rbar = 0.5 * (R - M + math.sqrt(R * R - 2.0 * M * R))
    lq = ys[:, 3] + (math.log(Rbar / R) - ys[-1, 3])             # ln(rbar / r), matched at the surface
    rbar = rs * np.exp(lq)
    nu = ys[:, 2] + (0.5 * math.log(1.0 - 2.0 * M / R) - ys[-1, 2])
    p = np.maximum(ys[:, 1], 0.0)
    rho = (p / K) ** (1.0 / Gamma)
    psi = np.sqrt(np.where(rbar > 0, rs / np.where(rbar > 0, rbar, 1.0), np.exp(-lq[0])))
    psi[0] = math.exp(-0.5 * lq[0])
    out = dict(rbar=rbar, rho=rho, p=p, alpha=np.exp(nu), psi=psi, M=M, R=R, Rbar=Rbar, K=K, Gamma=Gamma)
    _TOV_CACHE[key] = out
    return out


def tov_fields(prof, rb):
    """rho, p, alpha, psi, dp/drbar at isotropic radii rb (array): interior by interpolation, exterior analytic."""
    inside = rb < prof["Rbar"]
    rr = np.minimum(rb, prof["Rbar"])
    rho = np.where(inside, np.interp(rr, prof["rbar"], prof["rho"]), 0.0)
    p = np.where(inside, np.interp(rr, prof["rbar"], prof["p"]), 0.0)
    dpdr = np.where(inside, np.interp(rr, prof["rbar"], np.gradient(prof["p"], prof["rbar"])), 0.0)
    M = prof["M"]
    rsafe = np.maximum(rb, 1e-300)
    psi = np.where(inside, np.interp(rr, prof["rbar"], prof["psi"]), 1.0 + M / (2.0 * rsafe))
    alpha = np.where(inside, np.interp(rr, prof["rbar"], prof["alpha"]), (1.0 - M / (2.0 * rsafe)) / (1.0 + M / (2.0 * rsafe)))
    return rho, p, alpha, psi, dpdr


def tov_profile_barotrope(key, p_of_rho, e_of_rho, dpdrho, rho_c, rho_surf, dr=2.0e-3):
    """The same TOV equations as tov_profile for a general barotrope p(rho), e(rho) (total energy density), integrated in
    (m, rho, nu, ln(rbar/r)) with d rho/dr = (dp/dr) / (dp/drho) from the centre down to rho = rho_surf (the stellar surface of
    the synthetic star: the density below which the patch holds atmosphere). Initial data only; `key` caches the result."""
    if key in _TOV_CACHE:
        return _TOV_CACHE[key]

    def rhs(r, y):
        m, rho, nu, lq = y
        if r == 0.0:
            return np.array([0.0, 0.0, 0.0, 0.0])
        rho = max(rho, 0.5 * rho_surf)
        p, e = p_of_rho(rho), e_of_rho(rho)
        a = (m + 4.0 * math.pi * r ** 3 * p) / (r * (r - 2.0 * m))
        return np.array([4.0 * math.pi * r * r * e, -(e + p) * a / dpdrho(rho), a, (1.0 / math.sqrt(1.0 - 2.0 * m / r) - 1.0) / r])

    y = np.array([0.0, rho_c, 0.0, 0.0])
    r = 0.0
    rs, ys = [r], [y.copy()]
    while r < 100.0:
        k1 = rhs(r, y)
        k2 = rhs(r + 0.5 * dr, y + 0.5 * dr * k1)
        k3 = rhs(r + 0.5 * dr, y + 0.5 * dr * k2)
        k4 = rhs(r + dr, y + dr * k3)
        yn = y + dr / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
        if yn[1] <= rho_surf:                    # last partial step to the surface by linear interpolation in rho
            f = (y[1] - rho_surf) / (y[1] - yn[1])
            yn = y + f * (yn - y)
            r += f * dr
            yn[1] = rho_surf
            rs.append(r)
            ys.append(yn)
            break
        r += dr
        y = yn
        rs.append(r)
        ys.append(y.copy())
    rs, ys = np.array(rs), np.array(ys)
    M, R = ys[-1, 0], rs[-1]
    Rbar = 0.5 * (R - M + math.sqrt(R * R - 2.0 * M * R))
    lq = ys[:, 3] + (math.log(Rbar / R) - ys[-1, 3])
    rbar = rs * np.exp(lq)
    nu = ys[:, 2] + (0.5 * math.log(1.0 - 2.0 * M / R) - ys[-1, 2])
    rho = ys[:, 1]
    p = np.array([p_of_rho(x) for x in rho])
    psi = np.sqrt(np.where(rbar > 0, rs / np.where(rbar > 0, rbar, 1.0), np.exp(-lq[0])))
    psi[0] = math.exp(-0.5 * lq[0])
    out = dict(rbar=rbar, rho=rho, p=p, alpha=np.exp(nu), psi=psi, M=M, R=R, Rbar=Rbar)
    _TOV_CACHE[key] = out
    return out


# ---- config 3: static magnetised TOV star (BASELINE.json configs[2]) --------------------------------------
def config3(n=128, half_width=16.0, ng=NG, b_scale=1e-4, seed=SEED_BASE + 3):
    """Polytrope K=100, Gamma=2, rho_c=1.28e-3 (M ~ 1.4) on an n^3 patch of the given half width, outflow boundaries.
    gamma~_ij = delta_ij, chi = psi^-4, K_ij = 0, beta = 0, alpha from the TOV solution. Poloidal field from
    A_phi = A0 max(P - 0.04 P_max, 0) varpi^2, i.e. Bbar = curl(A) (the densitised field IS the flat curl), scaled so
    that max |B| = b_scale sqrt(P_max). Atmosphere rho = 1e-10 outside. Ideal gas Gamma = 2 (identical to the hybrid
    EoS with one piece and Gamma_th = Gamma)."""
    K, Gamma, rho_c = 100.0, 2.0, 1.28e-3
    prof = tov_profile(K, Gamma, rho_c)
    dx = 2.0 * half_width / n
    x0 = -half_width + 0.5 * dx
    X, Y, Z = mesh(n, n, n, ng, dx, x0=(x0, x0, x0))
    rb = np.sqrt(X * X + Y * Y + Z * Z)
    rho, p, alpha, psi, dpdr = tov_fields(prof, rb)
    par = default_params(eos_gamma=Gamma, rho_atmo=1e-10, rho_cut=1.01e-10, rho_low=1e-8)
    U = _flat_state(X.shape)
    U[CHI] = psi ** -4
    U[ALPHA] = alpha
    # conformally flat: Gamma~^i = 0, A~_ij = 0, K = 0
    P = np.zeros((NPRIM,) + X.shape)
    star = rho > 10.0 * par["rho_atmo"]
    P[RHO] = np.where(star, rho, par["rho_atmo"])
    P[EPS] = np.where(star, K * np.maximum(rho, 1e-300) ** (Gamma - 1.0) / (Gamma - 1.0), par["eps_atmo"])
    P[YE] = par["ye_atmo"]
    # vector potential A_x = -y Ab, A_y = x Ab, Ab = max(P - Pcut, 0):  Bbar = curl A
    pmax = K * rho_c ** Gamma
    on = p > 0.04 * pmax
    Ab = np.where(on, p - 0.04 * pmax, 0.0)
    dAb = np.where(on, dpdr, 0.0) / np.maximum(rb, 1e-300)       # (1/rbar) dAb/drbar, so that d_i Ab = x_i * dAb
    Bx, By, Bz = -X * Z * dAb, -Y * Z * dAb, 2.0 * Ab + (X * X + Y * Y) * dAb
    bmag = np.sqrt(Bx * Bx + By * By + Bz * Bz) * psi ** -4      # |B| = psi^-4 |Bbar|_flat
    scale = b_scale * math.sqrt(pmax) / bmag.max() if bmag.max() > 0 else 0.0
    U[BXBAR], U[BXBAR + 1], U[BXBAR + 2] = scale * Bx, scale * By, scale * Bz
    frac = float(star[ng:-ng, ng:-ng, ng:-ng].mean())
    return dict(U=U, P=P, n=(n, n, n), ng=ng, dx=dx, bc=[1] * 6, params=par, star_fraction=frac, tov=prof)


# ---- config 4: hot rotating magnetised star with a synthetic tabulated EoS (BASELINE.json configs[3]) --------
RHO_CGS_TO_CODE = 1.6199e-18          # G^3 Msun^2 / c^6 in cm^3 / g
_TABLE_CACHE = {}


def table_eos_analytic(rho, T, ye, K=2800.0, Gamma=2.5, gamma_th=1.75, cT=1.0e-3):
    """The closed form the synthetic table is filled from (input recipe, not method arithmetic):
    eps = K rho^(Gamma-1)/(Gamma-1) + cT T (1 + 0.2 (ye - 0.3)),  p = K rho^Gamma + (gamma_th - 1) rho eps_th,
    cs2 = (dp/drho|eps + p/rho^2 dp/deps|rho) / h  (a one-piece hybrid EoS). rho in code units, T in MeV."""
    eth = cT * T * (1.0 + 0.2 * (ye - 0.3))
    ec = K * rho ** (Gamma - 1.0) / (Gamma - 1.0)
    pc = K * rho ** Gamma
    p = pc + (gamma_th - 1.0) * rho * eth
    eps = ec + eth
    h = 1.0 + eps + p / rho
    dpdrho = Gamma * pc / rho + (gamma_th - 1.0) * eth - (gamma_th - 1.0) * pc / rho
    cs2 = (dpdrho + p / (rho * rho) * (gamma_th - 1.0) * rho) / h
    return p, eps, cs2


def make_table(n_rho=180, n_T=120, n_ye=50):
    """3-D table on (log10 rho[g/cc] in [3,16], log10 T[MeV] in [-1,2.3], Ye in [0.05,0.6]), rho fastest, then T, then Ye;
    columns log10 p, log10(eps + shift), cs2. The density axis is stored in code units (log10 rho_cgs + log10 1.6199e-18)."""
    key = (n_rho, n_T, n_ye)
    if key in _TABLE_CACHE:
        return _TABLE_CACHE[key]
    lr = np.linspace(3.0, 16.0, n_rho) + math.log10(RHO_CGS_TO_CODE)
    lT = np.linspace(-1.0, 2.3, n_T)
    ye = np.linspace(0.05, 0.6, n_ye)
    YE, LT, LR = np.meshgrid(ye, lT, lr, indexing="ij")
    p, eps, cs2 = table_eos_analytic(10.0 ** LR, 10.0 ** LT, YE)
    shift = 0.0
    tab = dict(n_rho=n_rho, n_T=n_T, n_ye=n_ye, lr0=lr[0], dlr=lr[1] - lr[0], lT0=lT[0], dlT=lT[1] - lT[0],
               ye0=ye[0], dye=ye[1] - ye[0], tab_eps_shift=shift, tab_h0=1.0,
               logp=np.ascontiguousarray(np.log10(p)), loge=np.ascontiguousarray(np.log10(eps + shift)),
               cs2=np.ascontiguousarray(np.minimum(cs2, 0.999)))
    _TABLE_CACHE[key] = tab
    return tab


def config4_thermal(rho, rho_c, T_star, T_floor=0.2):
    """Temperature [MeV] and electron fraction of the synthetic hot star as functions of density (input recipe): T falls from
    T_star at the centre to T_floor (inside the table, above its lower edge) like rho^(Gamma-1), Ye from 0.3 to 0.1."""
    x = np.maximum(rho, 0.0) / rho_c
    return T_floor + (T_star - T_floor) * x ** 1.5, 0.1 + 0.2 * x ** 0.25


def config4(n=256, ng=NG, seed=SEED_BASE + 4, table_shape=(180, 120, 50), T_star=10.0, v_eq=0.2, b_scale=1e-4):
    """Hot, rigidly rotating, magnetised star on an n^3 patch with the tabulated EoS (eos_kind = 2).
    Cold part p = K rho^2.5 with K = 2800 (gives p_c close to the Gamma = 2, K = 100 polytrope at rho_c = 1.28e-3); thermal part
    with T(rho), Ye(rho) of config4_thermal (T_star at the centre). The star is the TOV solution of THAT hot barotrope
    p(rho) = p_table(rho, T(rho), Ye(rho)) in isotropic coordinates, so the thermal pressure is in hydrostatic balance (a cold
    profile with a uniform temperature painted on is not: its surface layers, where the thermal pressure dominates, blow off
    and shock-heat past the table's eps_max, which the error policy of PAPER.md:1158-1162 treats as fatal);
    rigid rotation about z with Omega such that v = v_eq at the equator; poloidal field as in config 3; density
    multiplied by (1 + 1e-3 U(-1,1)) cell by cell (seeded). The patch width is Rbar / 0.46 (half width Rbar / 0.92), so that about 41 %
    of the cells are star."""
    Kc, Gc, rho_c = 2800.0, 2.5, 1.28e-3
    tab = make_table(*table_shape)
    # rho_low (R10, the "low-density region" of PAPER.md:1160-1162 where eps / v / Ye excursions are repaired instead of being
    # fatal) = 10 x the surface density of the synthetic star: the three-decade jump to the atmosphere makes the ratio
    # Dbar Ye / Dbar of the cells the surface spills into leave the table's Ye range
    par = default_params(eos_kind=2, rho_atmo=1e-10, rho_cut=1.01e-10, rho_low=1e-6, T_atmo=0.1, ye_min=0.05, ye_max=0.6,
                         ye_atmo=0.3, rho_max=10.0 ** (tab["lr0"] + tab["dlr"] * (tab["n_rho"] - 1)), eps_max=1e3)
    rho_surf = 1e3 * par["rho_atmo"]

    def p_of_rho(r):
        T, ye = config4_thermal(r, rho_c, T_star)
        return float(table_eos_analytic(r, T, ye, K=Kc, Gamma=Gc)[0])

    def e_of_rho(r):
        T, ye = config4_thermal(r, rho_c, T_star)
        return float(r * (1.0 + table_eos_analytic(r, T, ye, K=Kc, Gamma=Gc)[1]))

    def dpdrho(r):
        h = 1e-6 * r
        return (p_of_rho(r + h) - p_of_rho(r - h)) / (2.0 * h)

    prof = tov_profile_barotrope(("c4hot", Kc, Gc, rho_c, T_star, rho_surf), p_of_rho, e_of_rho, dpdrho, rho_c, rho_surf)
    half = prof["Rbar"] / 0.92
    dx = 2.0 * half / n
    x0 = -half + 0.5 * dx
    X, Y, Z = mesh(n, n, n, ng, dx, x0=(x0, x0, x0))
    rb = np.sqrt(X * X + Y * Y + Z * Z)
    rho, p, alpha, psi, dpdr = tov_fields(prof, rb)
    U = _flat_state(X.shape)
    U[CHI] = psi ** -4
    U[ALPHA] = alpha
    rng = SplitMix64(seed)
    noise = np.array([rng.uniform(-1.0, 1.0) for _ in range(4096)])
    idx = (np.arange(X.size, dtype=np.int64) * 2654435761 % 4096).reshape(X.shape)        # cheap seeded scatter of 4096 draws
    star = rho >= rho_surf
    P = np.zeros((NPRIM,) + X.shape)
    P[RHO] = np.where(star, rho * (1.0 + 1e-3 * noise[idx]), par["rho_atmo"])
    Ts, yes = config4_thermal(rho, rho_c, T_star)
    P[YE] = np.where(star, yes, par["ye_atmo"])
    Tf = np.where(star, Ts, par["T_atmo"])
    P[EPS] = table_eos_analytic(P[RHO], Tf, P[YE], K=Kc, Gamma=Gc)[1]
    # atmosphere eps must be what the EoS returns for T_atmo through the table (interpolated), the kernels reset it anyway
    omega = v_eq / prof["Rbar"]
    P[VX] = np.where(star, -omega * Y, 0.0)
    P[VX + 1] = np.where(star, omega * X, 0.0)
    pmax = p_of_rho(rho_c)
    on = p > 0.04 * pmax
    Ab = np.where(on, p - 0.04 * pmax, 0.0)
    dAb = np.where(on, dpdr, 0.0) / np.maximum(rb, 1e-300)
    Bx, By, Bz = -X * Z * dAb, -Y * Z * dAb, 2.0 * Ab + (X * X + Y * Y) * dAb
    bmag = np.sqrt(Bx * Bx + By * By + Bz * Bz) * psi ** -4
    scale = b_scale * math.sqrt(pmax) / bmag.max() if bmag.max() > 0 else 0.0
    U[BXBAR], U[BXBAR + 1], U[BXBAR + 2] = scale * Bx, scale * By, scale * Bz
    frac = float(star[ng:-ng, ng:-ng, ng:-ng].mean())
    return dict(U=U, P=P, n=(n, n, n), ng=ng, dx=dx, bc=[1] * 6, params=par, table=tab, star_fraction=frac, tov=prof)


def config1_tiled(n, **kw):
    """Config 1 at n > 32: the periodic 32^3 box tiled to n^3 at the same spacing (every field stays smooth and periodic
    when n is a multiple of 32; otherwise the wrap is a smooth-data jump the limiter handles). Bench workload c1_<n>."""
    base = config1(n=min(n, 32), **kw)
    if n <= 32:
        return base
    reps = (n + 31) // 32
    ng = base["ng"]

    def tile(A):
        inner = A[:, ng:-ng, ng:-ng, ng:-ng]
        big = np.tile(inner, (1, reps, reps, reps))[:, :n, :n, :n]
        return np.ascontiguousarray(np.pad(big, ((0, 0), (ng, ng), (ng, ng), (ng, ng)), mode="wrap"))
    base["U"], base["P"] = tile(base["U"]), tile(base["P"])
    base["n"] = (n, n, n)
    return base


# ---- config 5: two-star binary-like state + grey M1, 3 species (BASELINE.json configs[4]) ----------------------
NM1 = 15


def config5(n=192, half_width=60.0, separation=45.0, ng=NG, kappa0=1e-6, e_scale=1e-3, crop_on_star=False):
    """Two Gamma = 2, K = 100, rho_c = 1.28e-3 TOV stars at x = +-separation/2 with Newtonian circular-orbit velocities
    (+-v along y), conformal factors, lapses and a boost-like shift superposed (psi = 1 + sum (psi_i - 1),
    alpha = 1 + sum (alpha_i - 1), beta = - sum v_i (1 - alpha_i)); conformally flat, K_ij = 0. Three neutrino species
    with E = e_scale * scale_s * T^4 (T = p / rho, R27) inside the stars and a floor outside, F_i = 0, N = E.
    crop_on_star: the patch is centred on one star and n * dx covers 2.2 stellar radii (about 40 % star), the variant
    SURVEY.md 8(d) asks for so that the stiff-core path is exercised."""
    K, Gamma, rho_c = 100.0, 2.0, 1.28e-3
    prof = tov_profile(K, Gamma, rho_c)
    if crop_on_star:
        half_width = prof["Rbar"] / 0.92
        centre = (0.5 * separation, 0.0, 0.0)
    else:
        centre = (0.0, 0.0, 0.0)
    dx = 2.0 * half_width / n
    x0 = tuple(c - half_width + 0.5 * dx for c in centre)
    X, Y, Z = mesh(n, n, n, ng, dx, x0=x0)
    vorb = 0.5 * math.sqrt(2.0 * prof["M"] / separation)
    par = default_params(eos_gamma=Gamma, rho_atmo=1e-10, rho_cut=1.01e-10, rho_low=1e-8, m1_kappa0=kappa0)
    psi, alpha = np.ones_like(X), np.ones_like(X)
    beta = [np.zeros_like(X) for _ in range(3)]
    rho, vy = np.zeros_like(X), np.zeros_like(X)
    for sgn in (+1.0, -1.0):
        rb = np.sqrt((X - sgn * 0.5 * separation) ** 2 + Y * Y + Z * Z)
        r_, p_, a_, ps_, _ = tov_fields(prof, rb)
        psi += ps_ - 1.0
        alpha += a_ - 1.0
        beta[1] += -sgn * vorb * (1.0 - a_)
        rho += r_
        vy += np.where(r_ > 0.0, sgn * vorb, 0.0)
    U = _flat_state(X.shape)
    U[CHI] = psi ** -4
    U[ALPHA] = alpha
    for i in range(3):
        U[BETAX + i] = beta[i]
    star = rho > 10.0 * par["rho_atmo"]
    P = np.zeros((NPRIM,) + X.shape)
    P[RHO] = np.where(star, rho, par["rho_atmo"])
    P[EPS] = np.where(star, K * np.maximum(rho, 1e-300) ** (Gamma - 1.0) / (Gamma - 1.0), par["eps_atmo"])
    P[YE] = par["ye_atmo"]
    P[VX + 1] = np.where(star, vy, 0.0)
    U[BXBAR + 2] = 1e-6 * np.where(star, rho / rho_c, 0.0)
    T = np.where(star, (Gamma - 1.0) * P[EPS], 0.0)                 # T = p / rho for the ideal gas
    V = np.zeros((NM1,) + X.shape)
    sg = psi ** 6
    for s in range(3):
        E = np.maximum(e_scale * par["m1_species_scale"][s] * T ** 4, 1e-20)
        V[5 * s] = sg * E
        V[5 * s + 1] = sg * E
    frac = float(star[ng:-ng, ng:-ng, ng:-ng].mean())
    return dict(U=U, P=P, V=V, n=(n, n, n), ng=ng, dx=dx, bc=[1] * 6, params=par, star_fraction=frac, tov=prof)
