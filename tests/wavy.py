"""Test-side exact solutions used to pin the oracle (no oracle or CUDA code in here).

Minkowski spacetime in "wavy" coordinates: inertial X^M = x^M + a^M(x), a^M smooth and periodic in
space. g_mu_nu = eta_MN J^M_mu J^N_nu with J = d X / d x. This is an exact vacuum solution with a
non-trivial lapse, shift, 3-metric and extrinsic curvature, all depending on (t,x,y,z); adding a
Killing covector Z_M = c_M + w_MN X^N (w antisymmetric) gives an exact Z4 solution with Theta, Z_i != 0
(kappa_z = 0). A uniform boosted magnetised fluid in the inertial frame gives an exact solution of
the GRMHD equations (Eq. 32) on that background.
"""
import math

import numpy as np

from paper_2510_13965_b200 import synth

ETA = np.diag([-1.0, 1.0, 1.0, 1.0])

# a^M = AMP[M] * f(K[M] . x + PH[M]); spatial wavenumbers are integers (periodic box of side 2 pi)
AMP = [0.05, 0.04, 0.035, 0.03]
KVEC = [(-0.7, 1.0, 1.0, 1.0), (0.3, 1.0, -1.0, 0.0), (0.5, 1.0, 1.0, -1.0), (-0.4, 0.0, 1.0, 1.0)]
PH = [0.0, 0.4, 1.1, 2.3]
FUN = [(np.sin, np.cos, lambda p: -np.sin(p)), (np.cos, lambda p: -np.sin(p), lambda p: -np.cos(p)),
       (np.sin, np.cos, lambda p: -np.sin(p)), (np.cos, lambda p: -np.sin(p), lambda p: -np.cos(p))]
# Killing covector of Minkowski
ZC = np.array([0.05, -0.03, 0.04, 0.02])
ZW = np.zeros((4, 4))
for (m, n, val) in ((0, 1, 0.03), (0, 2, -0.02), (0, 3, 0.01), (1, 2, 0.025), (1, 3, -0.015), (2, 3, 0.02)):
    ZW[m, n], ZW[n, m] = val, -val


def _jac(t, X, Y, Z):
    """X^M, J^M_mu and dJ^M_mu/dx^lam at the grid points."""
    xs = [t + 0.0 * X, X, Y, Z]
    XM, J, dJ = [], [[None] * 4 for _ in range(4)], [[[None] * 4 for _ in range(4)] for _ in range(4)]
    for M in range(4):
        ph = sum(KVEC[M][mu] * xs[mu] for mu in range(4)) + PH[M]
        f0, f1, f2 = FUN[M][0](ph), FUN[M][1](ph), FUN[M][2](ph)
        XM.append(xs[M] + AMP[M] * f0)
        for mu in range(4):
            J[M][mu] = (1.0 if M == mu else 0.0) + AMP[M] * KVEC[M][mu] * f1
            for lam in range(4):
                dJ[M][mu][lam] = AMP[M] * KVEC[M][mu] * KVEC[M][lam] * f2
    return XM, J, dJ


def adm(t, X, Y, Z, with_Z=False):
    """gamma_ij, d_k gamma_ij, K_ij, alpha, beta^i (+ Theta, Z^i) of the wavy Minkowski slice at time t."""
    XM, J, dJ = _jac(t, X, Y, Z)
    g = [[sum(ETA[M, M] * J[M][mu] * J[M][nu] for M in range(4)) for nu in range(4)] for mu in range(4)]
    dg = [[[sum(ETA[M, M] * (dJ[M][mu][lam] * J[M][nu] + J[M][mu] * dJ[M][nu][lam]) for M in range(4))
            for lam in range(4)] for nu in range(4)] for mu in range(4)]      # dg[mu][nu][lam] = d_lam g_mu_nu
    gam = [[g[i + 1][j + 1] for j in range(3)] for i in range(3)]
    gi, det = synth._inv3(gam)
    bl = [g[0][i + 1] for i in range(3)]
    bu = [sum(gi[i][j] * bl[j] for j in range(3)) for i in range(3)]
    alpha = np.sqrt(sum(bu[i] * bl[i] for i in range(3)) - g[0][0])
    dgam = [[[dg[i + 1][j + 1][k + 1] for j in range(3)] for i in range(3)] for k in range(3)]   # [k][i][j]
    dtgam = [[dg[i + 1][j + 1][0] for j in range(3)] for i in range(3)]
    # d_i beta^k = -gamma^ka d_i gamma_ab beta^b + gamma^kj d_i g_0j
    dbu = [[sum(-gi[k][a] * dgam[i][a][b] * bu[b] for a in range(3) for b in range(3))
            + sum(gi[k][j] * dg[0][j + 1][i + 1] for j in range(3)) for k in range(3)] for i in range(3)]   # [i][k]
    Kij = [[None] * 3 for _ in range(3)]
    for i in range(3):
        for j in range(3):
            lie = sum(bu[k] * dgam[k][i][j] + gam[k][j] * dbu[i][k] + gam[i][k] * dbu[j][k] for k in range(3))
            Kij[i][j] = -(dtgam[i][j] - lie) / (2.0 * alpha)
    out = dict(gam=gam, dgam=dgam, Kij=Kij, alpha=alpha, beta=bu, J=J, gi=gi, det=det)
    if with_Z:
        ZM = [ZC[M] + sum(ZW[M, N] * XM[N] for N in range(4)) for M in range(4)]
        Zmu = [sum(J[M][mu] * ZM[M] for M in range(4)) for mu in range(4)]
        out["theta"] = -(Zmu[0] - sum(bu[i] * Zmu[i + 1] for i in range(3))) / alpha
        out["Zup"] = [sum(gi[i][j] * Zmu[j + 1] for j in range(3)) for i in range(3)]
    return out


def ccz4_fields(t, X, Y, Z, with_Z=False):
    a = adm(t, X, Y, Z, with_Z)
    return synth.conformal_from_adm(a["gam"], a["dgam"], a["Kij"], a["alpha"], a["beta"],
                                    a.get("theta"), a.get("Zup"))


def ddt(fun, t, h=2e-3):
    """6th-order centred time derivative of an array-valued function of t."""
    return (45.0 * (fun(t + h) - fun(t - h)) - 9.0 * (fun(t + 2 * h) - fun(t - 2 * h))
            + (fun(t + 3 * h) - fun(t - 3 * h))) / (60.0 * h)


# ---- uniform boosted magnetised fluid in the inertial frame ----------------------------------------
RHO0, EPS0 = 1.0e-3, 0.2
_vM = np.array([0.3, -0.2, 0.1])
_W0 = 1.0 / math.sqrt(1.0 - _vM @ _vM)
UM = np.concatenate([[_W0], _W0 * _vM])                   # u^M
_Bin = np.array([0.02, 0.03, -0.01])                      # inertial-frame B^I
# b^M with b.u = 0:  b^0 = W (B.v),  b^I = B^I / W + b^0 v^I
_b0 = _W0 * (_Bin @ _vM)
BM = np.concatenate([[_b0], _Bin / _W0 + _b0 * _vM])


def fluid(t, X, Y, Z):
    """coordinate-basis primitives (v^i, W) and Eulerian magnetic field B^i on the wavy slice at time t."""
    a = adm(t, X, Y, Z)
    J = a["J"]
    shape = X.shape
    Jm = np.zeros(shape + (4, 4))
    for M in range(4):
        for mu in range(4):
            Jm[..., M, mu] = J[M][mu]
    Ji = np.linalg.inv(Jm)                                # (J^-1)^mu_M
    u = np.einsum("...mM,M->...m", Ji, UM)                # u^mu
    b = np.einsum("...mM,M->...m", Ji, BM)
    alpha, beta = a["alpha"], a["beta"]
    W = alpha * u[..., 0]
    v = [u[..., i + 1] / W + beta[i] / alpha for i in range(3)]
    B = [W * b[..., i + 1] - alpha * b[..., 0] * u[..., i + 1] for i in range(3)]
    return a, v, W, B


# ---- radiation fields with a uniform stress-energy tensor in the inertial frame -------------------------
def radiation(t, X, Y, Z, TMN, NM):
    """Densitised M1 fields (Nbar, Ebar, Fbar_i) on the wavy slice at time t of a radiation field whose stress-energy tensor
    T^MN and number current N^M are CONSTANT in the inertial frame (so nabla_a T^ab = 0 and nabla_a N^a = 0 hold exactly):
    E = n_a n_b T^ab = alpha^2 T^tt, F_i = -n_a gamma_ib T^ab = alpha g_i_nu T^t_nu, N = -n_a N^a = alpha N^t (Eq. 35)."""
    a = adm(t, X, Y, Z)
    J = a["J"]
    shape = X.shape
    Jm = np.zeros(shape + (4, 4))
    for M in range(4):
        for mu in range(4):
            Jm[..., M, mu] = J[M][mu]
    Ji = np.linalg.inv(Jm)                                # (J^-1)^mu_M
    T = np.einsum("...mM,...nN,MN->...mn", Ji, Ji, TMN)   # T^mu_nu in wavy coordinates
    Nu = np.einsum("...mM,M->...m", Ji, NM)
    g = np.einsum("M,...Mm,...Mn->...mn", np.diag(ETA), Jm, Jm)
    alpha = a["alpha"]
    sg = np.sqrt(a["det"])
    E = alpha ** 2 * T[..., 0, 0]
    F = [alpha * np.einsum("...n,...n->...", g[..., i + 1, :], T[..., 0, :]) for i in range(3)]
    return np.stack([sg * alpha * Nu[..., 0], sg * E] + [sg * f for f in F])


def isotropic_radiation(J0, n0):
    """T^MN = 4/3 J u^M u^N + J/3 eta^MN, N^M = n u^M: radiation isotropic in the frame of the uniform fluid of `fluid`."""
    return 4.0 / 3.0 * J0 * np.outer(UM, UM) + J0 / 3.0 * ETA, n0 * UM


def null_beam(e0, n0, direction):
    """T^MN = e k^M k^N, N^M = n k^M with k = (1, unit vector): a single beam of free-streaming radiation."""
    d = np.asarray(direction, dtype=float)
    k = np.concatenate([[1.0], d / np.linalg.norm(d)])
    return e0 * np.outer(k, k), n0 * k
