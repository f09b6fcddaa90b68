// ORACLE (test infrastructure) — CCZ4 + gauge right-hand side, Sec. II A
// Eqs. (13)-(26) l.141-202, with the finite differences of Sec. III B and KO dissipation.
// Index loops follow the printed tensor expressions term by term.
#include <cmath>
#include "orc.hpp"

namespace orc {

static const int SYM[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};

// S_ij of PAPER.md:260 from the primitives, S_i (covariant, undensitised) and B^i
void stress_tensor(const double gl[3][3], const double vu[3], double W, double p,
                   const double Sl[3], const double Bu[3], double Sij[3][3]) {
  double vl[3], Bl[3];
  for (int i = 0; i < 3; ++i) {
    vl[i] = 0; Bl[i] = 0;
    for (int j = 0; j < 3; ++j) { vl[i] += gl[i][j] * vu[j]; Bl[i] += gl[i][j] * Bu[j]; }
  }
  double B2 = 0, Bv = 0;
  for (int i = 0; i < 3; ++i) { B2 += Bu[i] * Bl[i]; Bv += Bu[i] * vl[i]; }
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      Sij[i][j] = 0.5 * (vl[i] * Sl[j] + vl[j] * Sl[i]) + gl[i][j] * p
                  - 1.0 / (2.0 * W * W) * (2.0 * Bl[i] * Bl[j] - gl[i][j] * B2)
                  - 0.5 * Bv * (Bl[i] * vl[j] + Bl[j] * vl[i] - gl[i][j] * Bv);
}

void rhs_ccz4(const Params& par, const Grid& G, const double* U, const double* P, double* K) {
  const size_t n = G.npts();
  const long st[3] = {1, (long)G.mx(), (long)G.mx() * G.my()};
  const double hh[3] = {G.dx, G.dy, G.dz};
  const double PI = 3.14159265358979323846;
  const int ng = G.ng;
#pragma omp parallel for schedule(dynamic)
  for (int kk = ng; kk < G.nz + ng; ++kk)
  for (int jj = ng; jj < G.ny + ng; ++jj)
  for (int ii = ng; ii < G.nx + ng; ++ii) {
    const size_t p = G.idx(ii, jj, kk);
    auto F = [&](int f) { return U + (size_t)f * n + p; };
    // ---- fields at the point
    double g[3][3], A[3][3], Gh[3], be[3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { g[i][j] = *F(GXX + SYM[i][j]); A[i][j] = *F(AXX + SYM[i][j]); }
    const double chi = *F(CHI), Kh = *F(KHAT), Th = *F(THETA), al = *F(ALPHA);
    for (int i = 0; i < 3; ++i) { Gh[i] = *F(GAMX + i); be[i] = *F(BETAX + i); }
    // ---- centred derivatives, Eqs. (60)-(62)
    double d_g[3][3][3], d_chi[3], d_al[3], d_be[3][3], d_Kh[3], d_Th[3], d_Gh[3][3];
    double dd_g[3][3][3][3], dd_chi[3][3], dd_al[3][3], dd_be[3][3][3];
    auto D2 = [&](int f, int k, int l) {
      return k == l ? d2(F(f), st[k], hh[k]) : d11(F(f), st[k], hh[k], st[l], hh[l]);
    };
    for (int k = 0; k < 3; ++k) {
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) d_g[k][i][j] = d1(F(GXX + SYM[i][j]), st[k], hh[k]);
      d_chi[k] = d1(F(CHI), st[k], hh[k]);
      d_al[k] = d1(F(ALPHA), st[k], hh[k]);
      d_Kh[k] = d1(F(KHAT), st[k], hh[k]);
      d_Th[k] = d1(F(THETA), st[k], hh[k]);
      for (int i = 0; i < 3; ++i) { d_be[k][i] = d1(F(BETAX + i), st[k], hh[k]); d_Gh[k][i] = d1(F(GAMX + i), st[k], hh[k]); }
      for (int l = 0; l < 3; ++l) {
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) dd_g[k][l][i][j] = D2(GXX + SYM[i][j], k, l);
        dd_chi[k][l] = D2(CHI, k, l);
        dd_al[k][l] = D2(ALPHA, k, l);
        for (int i = 0; i < 3; ++i) dd_be[k][l][i] = D2(BETAX + i, k, l);
      }
    }
    // ---- inverse conformal metric (actual determinant; det gamma~ = 1 is not assumed)
    const double detg = g[0][0] * (g[1][1] * g[2][2] - g[1][2] * g[1][2]) - g[0][1] * (g[0][1] * g[2][2] - g[1][2] * g[0][2]) +
                        g[0][2] * (g[0][1] * g[1][2] - g[1][1] * g[0][2]);
    double gi[3][3];
    gi[0][0] = (g[1][1] * g[2][2] - g[1][2] * g[1][2]) / detg;
    gi[0][1] = gi[1][0] = (g[0][2] * g[1][2] - g[0][1] * g[2][2]) / detg;
    gi[0][2] = gi[2][0] = (g[0][1] * g[1][2] - g[0][2] * g[1][1]) / detg;
    gi[1][1] = (g[0][0] * g[2][2] - g[0][2] * g[0][2]) / detg;
    gi[1][2] = gi[2][1] = (g[0][1] * g[0][2] - g[0][0] * g[1][2]) / detg;
    gi[2][2] = (g[0][0] * g[1][1] - g[0][1] * g[0][1]) / detg;
    // ---- conformal Christoffels: Gl[k][i][j] = Gamma~_kij, Gu[k][i][j] = Gamma~^k_ij, Gt[k] = gamma~^ij Gamma~^k_ij (R5)
    double Gl[3][3][3], Gu[3][3][3], Gt[3], Z[3];
    for (int k = 0; k < 3; ++k) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j)
      Gl[k][i][j] = 0.5 * (d_g[i][k][j] + d_g[j][k][i] - d_g[k][i][j]);
    for (int k = 0; k < 3; ++k) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
      Gu[k][i][j] = 0;
      for (int l = 0; l < 3; ++l) Gu[k][i][j] += gi[k][l] * Gl[l][i][j];
    }
    for (int k = 0; k < 3; ++k) {
      Gt[k] = 0;
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Gt[k] += gi[i][j] * Gu[k][i][j];
      Z[k] = 0.5 * chi * (Gh[k] - Gt[k]);                  // PAPER.md:132  Gamma^ = Gamma~ + 2 Z / chi
    }
    // ---- Ricci pieces
    double Rh[3][3], cRc[3][3];
    double lapchi = 0, Ghdchi = 0;
    for (int k = 0; k < 3; ++k) {
      Ghdchi += Gh[k] * d_chi[k];
      for (int m = 0; m < 3; ++m) lapchi += gi[k][m] * (dd_chi[k][m] - 3.0 / (2.0 * chi) * d_chi[k] * d_chi[m]);
    }
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
      double r = 0;
      for (int m = 0; m < 3; ++m) for (int nn = 0; nn < 3; ++nn) r += -0.5 * gi[m][nn] * dd_g[m][nn][i][j];
      for (int k = 0; k < 3; ++k) r += 0.5 * (g[k][i] * d_Gh[j][k] + g[k][j] * d_Gh[i][k]);
      for (int k = 0; k < 3; ++k) r += 0.5 * Gh[k] * (Gl[i][j][k] + Gl[j][i][k]);
      for (int m = 0; m < 3; ++m) for (int nn = 0; nn < 3; ++nn) for (int k = 0; k < 3; ++k)
        r += gi[m][nn] * (Gu[k][m][i] * Gl[j][k][nn] + Gu[k][m][j] * Gl[i][k][nn] + Gu[k][m][i] * Gl[k][nn][j]);
      Rh[i][j] = r;                                                                     // Eq. (23)
      double c = 0.5 * dd_chi[i][j] - d_chi[i] * d_chi[j] / (4.0 * chi);
      for (int k = 0; k < 3; ++k) c += -0.5 * Gu[k][i][j] * d_chi[k];
      for (int k = 0; k < 3; ++k) c += (2.0 / chi) * Z[k] * 0.5 * (g[k][i] * d_chi[j] + g[k][j] * d_chi[i]);
      c += 0.5 * g[i][j] * (lapchi - Ghdchi);
      cRc[i][j] = c;                                                                    // chi R^chi_ij, Eq. (22)
    }
    // ---- D_i D_j alpha with physical Christoffels (R25)
    double DDal[3][3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
      double s = dd_al[i][j];
      for (int k = 0; k < 3; ++k) {
        double gdchi = 0;
        for (int l = 0; l < 3; ++l) gdchi += gi[k][l] * d_chi[l];
        const double Gp = Gu[k][i][j] - ((k == i ? d_chi[j] : 0.0) + (k == j ? d_chi[i] : 0.0) - g[i][j] * gdchi) / (2.0 * chi);
        s -= Gp * d_al[k];
      }
      DDal[i][j] = s;
    }
    // ---- matter projections (R6; tau_ADM = tau + D and S_i from the evolved fields, S_ij from l.260)
    double E = 0, Sl[3] = {0, 0, 0}, Sij[3][3] = {{0}}, Str = 0;
    if (par.grav_G != 0.0) {
      const double isg = chi * std::sqrt(chi);
      E = (*F(TAUBAR) + *F(DBAR)) * isg;
      double gl[3][3], vu[3], Bu[3];
      for (int i = 0; i < 3; ++i) {
        Sl[i] = *F(SXBAR + i) * isg; Bu[i] = *F(BXBAR + i) * isg; vu[i] = P[(size_t)(VX + i) * n + p];
        for (int j = 0; j < 3; ++j) gl[i][j] = g[i][j] / chi;
      }
      stress_tensor(gl, vu, P[(size_t)WLOR * n + p], P[(size_t)PRESS * n + p], Sl, Bu, Sij);
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Str += chi * gi[i][j] * Sij[i][j];
    }
    const double G8 = 8.0 * PI * par.grav_G;
    // ---- common contractions
    double divb = 0, trA = 0, Aud[3][3], Auu[3][3], AA = 0;
    for (int k = 0; k < 3; ++k) divb += d_be[k][k];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
      trA += gi[i][j] * A[i][j];                           // R4: A~ = gamma~^ij A~_ij
      Aud[i][j] = 0;
      for (int l = 0; l < 3; ++l) Aud[i][j] += gi[i][l] * A[l][j];
    }
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
      Auu[i][j] = 0;
      for (int l = 0; l < 3; ++l) Auu[i][j] += Aud[i][l] * gi[l][j];
      AA += Aud[i][j] * Aud[j][i];
    }
    auto adv = [&](int f) {
      double s = 0;
      for (int k = 0; k < 3; ++k) s += be[k] * dadv(F(f), st[k], hh[k], be[k]);
      return s;
    };
    auto ko = [&](int f) {
      double s = 0;
      for (int k = 0; k < 3; ++k) s += dko(F(f), st[k], hh[k], par.sigma_ko_spacetime);
      return s;
    };
    auto OUT = [&](int f) -> double& { return K[(size_t)f * n + p]; };
    // ---- Eq. (13)
    for (int i = 0; i < 3; ++i) for (int j = i; j < 3; ++j) {
      double s = adv(GXX + SYM[i][j]);
      for (int k = 0; k < 3; ++k) s += g[i][k] * d_be[j][k] + g[k][j] * d_be[i][k];
      s += -2.0 / 3.0 * g[i][j] * divb - 2.0 * al * (A[i][j] - g[i][j] * trA / 3.0) - al / 3.0 * par.kappa_c * g[i][j] * std::log(detg);
      OUT(GXX + SYM[i][j]) = s + ko(GXX + SYM[i][j]);
    }
    // ---- Eq. (14)
    double X[3][3], trX = 0;
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
      X[i][j] = al * (chi * Rh[i][j] + cRc[i][j] - G8 * chi * Sij[i][j]) - chi * DDal[i][j];
      trX += gi[i][j] * X[i][j];
    }
    for (int i = 0; i < 3; ++i) for (int j = i; j < 3; ++j) {
      double s = adv(AXX + SYM[i][j]);
      for (int k = 0; k < 3; ++k) s += A[i][k] * d_be[j][k] + A[k][j] * d_be[i][k];
      s += -2.0 / 3.0 * A[i][j] * divb - al / 3.0 * par.kappa_c * g[i][j] * trA;
      s += X[i][j] - g[i][j] * trX / 3.0;
      double AAij = 0;
      for (int k = 0; k < 3; ++k) AAij += A[i][k] * Aud[k][j];
      s += al * (Kh * A[i][j] - 2.0 * AAij);
      OUT(AXX + SYM[i][j]) = s + ko(AXX + SYM[i][j]);
    }
    // ---- Eq. (15)
    OUT(CHI) = adv(CHI) + 2.0 / 3.0 * chi * (al * (Kh + 2.0 * Th) - divb) + ko(CHI);
    // ---- Eq. (16) with Eq. (24)
    double lapal = 0, Zdal = 0;
    for (int i = 0; i < 3; ++i) {
      lapal -= chi * Gt[i] * d_al[i];
      Zdal += Z[i] * d_al[i];
      for (int j = 0; j < 3; ++j) lapal += chi * gi[i][j] * dd_al[i][j] - 0.5 * gi[i][j] * d_al[i] * d_chi[j];
    }
    const double Ktot = Kh + 2.0 * Th;
    OUT(KHAT) = adv(KHAT) - lapal + al * (Ktot * Ktot / 3.0 + AA + 0.5 * G8 * (E + Str) + par.kappa_z * (1.0 - par.kappa_2) * Th) + 2.0 * Zdal + ko(KHAT);
    // ---- Eq. (17)
    double Rtr = 0;
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Rtr += gi[i][j] * (chi * Rh[i][j] + cRc[i][j]);
    OUT(THETA) = adv(THETA) + 0.5 * al * (Rtr + 2.0 / 3.0 * Kh * Kh + 2.0 / 3.0 * Th * (Kh - 2.0 * Th) - AA) - Zdal
                 - al * (G8 * E + par.kappa_z * (2.0 + par.kappa_2) * Th) + ko(THETA);
    // ---- Eqs. (18)-(20)
    for (int i = 0; i < 3; ++i) {
      double s = adv(GAMX + i) + 2.0 / 3.0 * Gh[i] * divb;
      for (int j = 0; j < 3; ++j) {
        s -= Gh[j] * d_be[j][i];
        for (int k = 0; k < 3; ++k) s += gi[j][k] * dd_be[j][k][i] + gi[i][j] * dd_be[j][k][k] / 3.0;
        s -= 2.0 * Auu[i][j] * d_al[j];
      }
      double b1 = 0, b2 = 0;
      for (int j = 0; j < 3; ++j) {
        for (int k = 0; k < 3; ++k) b1 += Gu[i][j][k] * Auu[j][k];
        b1 += -3.0 / (2.0 * chi) * Auu[i][j] * d_chi[j] - 2.0 / 3.0 * gi[i][j] * d_Kh[j] - G8 * gi[i][j] * Sl[j];   // R7
        b2 += -gi[i][j] * (d_Th[j] / 3.0 + Th / al * d_al[j]);
      }
      b2 += -Z[i] / chi * (par.kappa_z + 2.0 / 3.0 * Ktot);
      OUT(GAMX + i) = s + 2.0 * al * b1 + 2.0 * al * b2 + ko(GAMX + i);
    }
    // ---- gauge, Eqs. (25)-(26)
    OUT(ALPHA) = adv(ALPHA) - 2.0 * al * par.f_alpha * Kh + ko(ALPHA);
    for (int i = 0; i < 3; ++i)
      OUT(BETAX + i) = adv(BETAX + i) + 0.75 * par.f_beta * Gh[i] - par.eta_shift * (be[i] - par.beta0[i]) + ko(BETAX + i);
  }
}

}  // namespace orc
