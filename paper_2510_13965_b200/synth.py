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
