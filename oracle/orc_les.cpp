// ORACLE (test infrastructure) — Large-Eddy-Simulation gradient sub-grid-scale terms: the tensor of the induction
// equation, C_M = par.les_C_M (the paper's production value is 8, l.863), and the other three of (A11), C_N, C_Y, C_T (zero in the paper's
// runs). PAPER.md Sec. II B l.252-256 and App. A, Eqs. (A11)-(A17) l.855-882, followed term by term in the paper's notation.
//
// Readings (R39-R47; the appendix uses symbols the paper does not define — they are fixed by the requirement that the
// printed chain (A12)-(A16) equals the gradient model the appendix itself states, tau_F^k = -xi grad(dF^k/dC) . grad C, which the
// pins check numerically: tests/test_oracle_les.py):
//   calE = h W^2 with h = rho (1 + eps) + p the enthalpy density (l.232);  Theta = calE + B^2 (so S_i = Theta v_i - (v.B) B_i, Eq. 29);
//   E^i = -eps^{ijk} v_j B_k (eps^{ijk} = [ijk]/sqrt(gamma)), E^2 = E_i E^i;  D = rho W;
//   grad f . grad g = gamma^{ij} d_i f d_j g with d_i the fourth-order centred difference of Eq. (60) applied to the FIELD f
//   (components v^k, B^k, v_k, B_k, E_k, E^k are differentiated as scalar fields; grad ln rho = grad rho / rho);
//   H_M^{ki}: the FIRST index is the flux direction (the k of d_k in Eq. 32; Eq. 32 prints G_B^{ik}, (A11)/(A16) print ^{ki}: the
//   filtered product rule  bar(fg) = bar f bar g + 2 xi grad f . grad g  of l.814 decides);
//   xi = gamma^{1/3} Delta^2 / 24 with Delta = (dx dy dz)^{1/3};
//   the SGS flux is part of the flux bracket of Eq. (32): it is added to the pointwise flux F^k of Bbar^i BEFORE the flux
//   splitting and reconstruction; it is evaluated at every grid point at least 2 points away from the array edge (ghost width >= 5
//   covers all nodes the reconstruction of interior interfaces touches), zero elsewhere.
#include <cmath>
#include <vector>
#include "orc.hpp"

namespace orc {

static const int SYM[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};

// the 29 auxiliary fields whose gradients App. A needs, at one point
void les_aux_point(const Params& par, const double gl[3][3], double sqrtg, const double Bu[3], const double prim[NPRIM], double a[LES_NAUX]) {
  const double rho = prim[RHO], eps = prim[EPS], p = prim[PRESS], W = prim[WLOR];
  double vu[3] = {prim[VX], prim[VY], prim[VZ]}, vl[3], Bl[3];
  for (int i = 0; i < 3; ++i) {
    vl[i] = 0.0; Bl[i] = 0.0;
    for (int j = 0; j < 3; ++j) { vl[i] += gl[i][j] * vu[j]; Bl[i] += gl[i][j] * Bu[j]; }
  }
  double vB = 0.0, B2 = 0.0;
  for (int i = 0; i < 3; ++i) { vB += vl[i] * Bu[i]; B2 += Bl[i] * Bu[i]; }
  // E^i = -eps^{ijk} v_j B_k,  eps^{ijk} = [ijk] / sqrt(gamma)
  double Eu[3], El[3];
  for (int i = 0; i < 3; ++i) {
    const int j = (i + 1) % 3, k = (i + 2) % 3;
    Eu[i] = -(vl[j] * Bl[k] - vl[k] * Bl[j]) / sqrtg;
  }
  for (int i = 0; i < 3; ++i) { El[i] = 0.0; for (int j = 0; j < 3; ++j) El[i] += gl[i][j] * Eu[j]; }
  const double h = rho * (1.0 + eps) + p;
  for (int i = 0; i < 3; ++i) {
    a[LES_BU + i] = Bu[i]; a[LES_VU + i] = vu[i]; a[LES_VL + i] = vl[i]; a[LES_BL + i] = Bl[i]; a[LES_EL + i] = El[i]; a[LES_EU + i] = Eu[i];
  }
  a[LES_VB] = vB;
  a[LES_TH] = h * W * W + B2;
  a[LES_WM2] = 1.0 / (W * W);
  a[LES_RHO] = rho; a[LES_EPS] = eps; a[LES_H] = h;
  eos_dp(par, rho, eps, prim[YE], a[LES_DPDRHO], a[LES_DPDEPS], a[LES_DPDYE]);
  a[LES_YE] = prim[YE];
  a[LES_D] = rho * W;
  a[LES_CALE] = h * W * W;
  a[LES_DYE] = rho * W * prim[YE];
}

// H_M^{ki} of Eq. (A16) at one point: a = auxiliary fields, da[m] = their partial derivatives d_m, gu = gamma^{ij}, p = pressure
// H_M^{ki} of (A16) and, when HN / HNY / HT are not null, H_N^k, H_{N_Y}^k of (A15) and H_T^{ki} of (A17) (both indices up) at one point:
// a = auxiliary fields, da[m] = their partial derivatives d_m, gu = gamma^{ij}, gl = gamma_ij, sqrtg = sqrt(gamma), p = pressure
void les_H_point(const double a[LES_NAUX], const double da[3][LES_NAUX], const double gu[3][3], const double gl[3][3], double sqrtg, double p,
                 double HM[3][3], double* HN, double* HNY, double (*HT)[3]) {
  auto dot = [&](int f, int g) {                              // grad f . grad g = gamma^{mn} d_m f d_n g
    double s = 0.0;
    for (int m = 0; m < 3; ++m) for (int n = 0; n < 3; ++n) s += gu[m][n] * da[m][f] * da[n][g];
    return s;
  };
  const double* Bu = a + LES_BU; const double* vu = a + LES_VU; const double* vl = a + LES_VL; const double* Bl = a + LES_BL;
  const double* El = a + LES_EL; const double* Eu = a + LES_EU;
  const double vB = a[LES_VB], Th = a[LES_TH], W2 = 1.0 / a[LES_WM2], rho = a[LES_RHO], h = a[LES_H];
  const double dpdrho = a[LES_DPDRHO], dpdeps = a[LES_DPDEPS];
  const double calE = h * W2;
  double E2 = 0.0;
  for (int j = 0; j < 3; ++j) E2 += El[j] * Eu[j];
  // ---- Psi_v^k (first line of A12)
  double sBv = 0.0, sBBvB = 0.0, sBvTh = 0.0;
  for (int j = 0; j < 3; ++j) {
    sBv += dot(LES_BU + j, LES_VL + j);                       // grad B^j . grad v_j
    sBBvB += Bl[j] * dot(LES_BU + j, LES_VB);                 // B_j grad B^j . grad (v.B)
    sBvTh += Bu[j] * dot(LES_VL + j, LES_TH);                 // B^j grad v_j . grad Theta
  }
  double Psi_v[3];
  for (int k = 0; k < 3; ++k)
    Psi_v[k] = 2.0 / Th * (dot(LES_VB, LES_BU + k) - dot(LES_TH, LES_VU + k) + Bu[k] / calE * (Th * sBv + sBBvB - sBvTh));
  // ---- Psi_M^{ki} (second line): X^{[i} Y^{k]} = (X^i Y^k - X^k Y^i) / 2
  double Psi_M[3][3];
  for (int k = 0; k < 3; ++k) for (int i = 0; i < 3; ++i) {
    const double t1 = 0.5 * (dot(LES_BU + i, LES_VU + k) - dot(LES_BU + k, LES_VU + i));
    const double t2 = 0.5 * (Bu[i] * dot(LES_BU + k, LES_VB) - Bu[k] * dot(LES_BU + i, LES_VB));
    const double t3 = 0.5 * (Bu[i] * dot(LES_VU + k, LES_TH) - Bu[k] * dot(LES_VU + i, LES_TH));
    Psi_M[k][i] = 4.0 / Th * (Th * t1 + t2 - t3);
  }
  // ---- Psi_Theta, Psi_A (third line)
  double sBB = 0.0, sEE = 0.0, svv = 0.0, BvPsi = 0.0;
  for (int j = 0; j < 3; ++j) {
    sBB += dot(LES_BL + j, LES_BU + j);                       // grad B_j . grad B^j
    sEE += dot(LES_EL + j, LES_EU + j);
    svv += dot(LES_VL + j, LES_VU + j);
  }
  for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) BvPsi += 0.5 * (Bl[i] * vl[k] - Bl[k] * vl[i]) * Psi_M[k][i];   // B_[i v_k] Psi_M^{ki}
  const double Psi_Th = Th / (Th - E2) * (sBB - sEE - BvPsi);
  const double Psi_A = W2 * (p * dpdeps + rho * rho * dpdrho);
  // ---- H_p (A12). The two Y_e terms are printed after the closing brace; the definition the appendix states (tau = -xi grad(dF/dC).grad C, checked
  // numerically with a Y_e-dependent EoS) puts them INSIDE the braces with the factor rho of the first term (reading R42): rho [grad(dp/dYe).grad Ye -
  // (2/D) dp/dYe grad Ye.grad D]
  double vPsi = 0.0;
  for (int j = 0; j < 3; ++j) vPsi += vl[j] * Psi_v[j];
  const double dWW = dot(LES_WM2, LES_WM2);
  const double pref = calE * W2 * (Th - E2) / ((rho * calE - Psi_A) * (Th - E2) * W2 + Psi_A * Th);
  const double brace =
      rho * (dot(LES_DPDRHO, LES_RHO) + dot(LES_DPDEPS, LES_EPS)) - 2.0 * dpdeps * dot(LES_RHO, LES_EPS)
      - (calE * dpdeps - Psi_A) * (0.25 * W2 * dWW + dot(LES_WM2, LES_RHO) / rho)
      - 2.0 / W2 * dpdeps * (sBB - W2 * W2 * dot(LES_WM2, LES_H))
      - (calE * dpdeps + Psi_A) * (vPsi + svv + W2 * dWW)
      + Psi_Th / (calE * Th) * ((calE * dpdeps + Psi_A) * (Th - E2) - Psi_A * Th / W2)
      + rho * (dot(LES_DPDYE, LES_YE) - 2.0 / a[LES_D] * a[LES_DPDYE] * dot(LES_YE, LES_D));
  const double H_p = pref * brace;
  const double H_Th = Psi_Th + Th / (Th - E2) * H_p;                                        // (A13)
  double H_v[3];
  for (int k = 0; k < 3; ++k) H_v[k] = Psi_v[k] - (vu[k] + vB / calE * Bu[k]) * H_Th / Th;  // (A14)
  for (int k = 0; k < 3; ++k) for (int i = 0; i < 3; ++i)                                   // (A16): 2 B^[i H_v^k] + 4 grad B^[i . grad v^k]
    HM[k][i] = (Bu[i] * H_v[k] - Bu[k] * H_v[i]) + 2.0 * (dot(LES_BU + i, LES_VU + k) - dot(LES_BU + k, LES_VU + i));
  if (HN) for (int k = 0; k < 3; ++k) HN[k] = 2.0 * dot(LES_D, LES_VU + k) + a[LES_D] * H_v[k];              // (A15)
  if (HNY) for (int k = 0; k < 3; ++k) HNY[k] = 2.0 * dot(LES_DYE, LES_VU + k) + a[LES_DYE] * H_v[k];
  if (HT) {
    // H_E^i = 1/2 eps^i_{jk} H_M^{jk} (A16) is the same contraction for E^i = -eps^{ijk} v_j B_k: with the FIRST index of H_M the flux direction (R40, R45),
    // H_M^{(dir k)(comp j)} belongs to the flux B^j v^k - B^k v^j, so that eps_{ijk} (B^j v^k - B^k v^j) / 2 = -eps_{ijk} v^j B^k = E_i and
    // H_E_i = 1/2 sqrt(gamma) [ijk] H_M^{(dir k)(comp j)}; E only enters (A17) quadratically, so its overall sign convention does not matter
    double HEl[3], HEu[3];
    for (int i = 0; i < 3; ++i) {
      const int j = (i + 1) % 3, k = (i + 2) % 3;
      HEl[i] = 0.5 * sqrtg * (HM[k][j] - HM[j][k]);
    }
    for (int i = 0; i < 3; ++i) { HEu[i] = 0.0; for (int j = 0; j < 3; ++j) HEu[i] += gu[i][j] * HEl[j]; }
    double EHE = 0.0;
    for (int j = 0; j < 3; ++j) EHE += El[j] * HEu[j];
    (void)gl;
    const double trace = H_p + sBB + sEE + EHE;
    for (int k = 0; k < 3; ++k) for (int i = 0; i < 3; ++i) {
      // grad calE . grad (v^k v^i) by the product rule (reading R46): v^k grad calE . grad v^i + v^i grad calE . grad v^k
      const double first = vu[k] * dot(LES_CALE, LES_VU + i) + vu[i] * dot(LES_CALE, LES_VU + k)
                           + calE * (0.5 * (vu[k] * H_v[i] + vu[i] * H_v[k]) + dot(LES_VU + k, LES_VU + i)) + vu[k] * vu[i] * H_p;
      const double second = dot(LES_BU + k, LES_BU + i) + dot(LES_EU + k, LES_EU + i) + 0.5 * (Eu[k] * HEu[i] + Eu[i] * HEu[k]);
      HT[k][i] = 2.0 * first - 2.0 * second + (gu[k][i] - vu[k] * vu[i]) * trace;                              // (A17)
    }
  }
}

void les_HM_point(const double a[LES_NAUX], const double da[3][LES_NAUX], const double gu[3][3], double p, double HM[3][3]) {
  const double id[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
  les_H_point(a, da, gu, id, 1.0, p, HM, nullptr, nullptr, nullptr);
}

// SGS parts of the flux brackets of Eq. (32) in direction k, -alpha G = +alpha C xi sqrt(gamma) H (A11), in the LES_NFLUX = 24 fields of L:
//   3 k + i       Bbar^i:  C_M H_M^{ki}            9 + k   Dbar: C_N H_N^k           12 + k   DYebar: C_Y H_{N_Y}^k
//   15 + 3 k + i  Sbar_i:  C_T gamma_ij H_T^{kj}   (taubar: (A11) defines no G_tau, none is added: reading R47)
// A (LES_NAUX fields) receives the auxiliary fields (for the pins)
void les_flux(const Params& par, const Grid& G, const double* U, const double* P, double* L, double* A) {
  const size_t n = G.npts();
  const long st[3] = {1, (long)G.mx(), (long)G.mx() * G.my()};
  const double hh[3] = {G.dx, G.dy, G.dz};
  const double Delta2 = std::pow(G.dx * G.dy * G.dz, 2.0 / 3.0);
  for (size_t q = 0; q < (size_t)LES_NFLUX * n; ++q) L[q] = 0.0;
  const bool full = par.les_C_N != 0.0 || par.les_C_Y != 0.0 || par.les_C_T != 0.0;
  // auxiliary fields at every grid point
  for (int kk = 0; kk < G.mz(); ++kk) for (int jj = 0; jj < G.my(); ++jj) for (int ii = 0; ii < G.mx(); ++ii) {
    const size_t p = G.idx(ii, jj, kk);
    const double chi = U[(size_t)CHI * n + p];
    double gl[3][3], Bu[3], prim[NPRIM], a[LES_NAUX];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) gl[i][j] = U[(size_t)(GXX + SYM[i][j]) * n + p] / chi;
    const double sqrtg = 1.0 / (chi * std::sqrt(chi));
    for (int i = 0; i < 3; ++i) Bu[i] = U[(size_t)(BXBAR + i) * n + p] / sqrtg;
    for (int f = 0; f < NPRIM; ++f) prim[f] = P[(size_t)f * n + p];
    les_aux_point(par, gl, sqrtg, Bu, prim, a);
    for (int f = 0; f < LES_NAUX; ++f) A[(size_t)f * n + p] = a[f];
  }
  // gradients (Eq. 60) and H_M wherever the stencil fits
#pragma omp parallel for schedule(dynamic)
  for (int kk = 2; kk < G.mz() - 2; ++kk) for (int jj = 2; jj < G.my() - 2; ++jj) for (int ii = 2; ii < G.mx() - 2; ++ii) {
    const size_t p = G.idx(ii, jj, kk);
    double a[LES_NAUX], da[3][LES_NAUX];
    for (int f = 0; f < LES_NAUX; ++f) {
      a[f] = A[(size_t)f * n + p];
      for (int m = 0; m < 3; ++m) da[m][f] = d1(A + (size_t)f * n + p, st[m], hh[m]);
    }
    const double chi = U[(size_t)CHI * n + p], al = U[(size_t)ALPHA * n + p];
    double g[3][3], gu[3][3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) g[i][j] = U[(size_t)(GXX + SYM[i][j]) * n + p];
    const double det = g[0][0] * (g[1][1] * g[2][2] - g[1][2] * g[1][2]) - g[0][1] * (g[0][1] * g[2][2] - g[1][2] * g[0][2]) +
                       g[0][2] * (g[0][1] * g[1][2] - g[1][1] * g[0][2]);
    gu[0][0] = chi * (g[1][1] * g[2][2] - g[1][2] * g[1][2]) / det;
    gu[0][1] = gu[1][0] = chi * (g[0][2] * g[1][2] - g[0][1] * g[2][2]) / det;
    gu[0][2] = gu[2][0] = chi * (g[0][1] * g[1][2] - g[0][2] * g[1][1]) / det;
    gu[1][1] = chi * (g[0][0] * g[2][2] - g[0][2] * g[0][2]) / det;
    gu[1][2] = gu[2][1] = chi * (g[0][1] * g[0][2] - g[0][0] * g[1][2]) / det;
    gu[2][2] = chi * (g[0][0] * g[1][1] - g[0][1] * g[0][1]) / det;
    double HM[3][3], HN[3], HNY[3], HT[3][3], gl[3][3];
    const double sqrtg = 1.0 / (chi * std::sqrt(chi));
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) gl[i][j] = g[i][j] / chi;
    les_H_point(a, da, gu, gl, sqrtg, P[(size_t)PRESS * n + p], HM, full ? HN : nullptr, full ? HNY : nullptr, full ? HT : nullptr);
    const double xi = Delta2 / (24.0 * chi);                  // gamma^{1/3} Delta^2 / 24, gamma = chi^-3
    const double fac = al * xi * sqrtg;
    for (int k = 0; k < 3; ++k) for (int i = 0; i < 3; ++i) L[(size_t)(3 * k + i) * n + p] = fac * par.les_C_M * HM[k][i];
    if (full)
      for (int k = 0; k < 3; ++k) {
        L[(size_t)(9 + k) * n + p] = fac * par.les_C_N * HN[k];
        L[(size_t)(12 + k) * n + p] = fac * par.les_C_Y * HNY[k];
        for (int i = 0; i < 3; ++i) {
          double lowered = 0.0;
          for (int j = 0; j < 3; ++j) lowered += gl[i][j] * HT[k][j];
          L[(size_t)(15 + 3 * k + i) * n + p] = fac * par.les_C_T * lowered;
        }
      }
  }
}

}  // namespace orc
