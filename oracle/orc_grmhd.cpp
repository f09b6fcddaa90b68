// ORACLE (test infrastructure) — GRMHD balance laws, Eq. (32) l.256-260, discretised with
// the Lax-Friedrichs flux splitting + MP5 of Sec. III C (Eqs. 63-76) and the speed bound of
// App. B (Eqs. B1-B3).
#include <algorithm>
#include <cmath>
#include <vector>
#include "orc.hpp"

namespace orc {

void stress_tensor(const double gl[3][3], const double vu[3], double W, double p,
                   const double Sl[3], const double Bu[3], double Sij[3][3]);

static const int SYM[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};

namespace {
struct Pt {   // everything the flux brackets of Eq. (32) need at one grid point
  double al, be[3], chi, g[3][3], gi[3][3];       // conformal metric and inverse
  double uc[10];                                  // densitised conserved fields
  double rho, eps, p, vu[3], W, cs2;
};
}

static void load_point(const Grid& G, const double* U, const double* P, size_t p, Pt& q) {
  const size_t n = G.npts();
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) q.g[i][j] = U[(size_t)(GXX + SYM[i][j]) * n + p];
  const double (*g)[3] = q.g;
  const double det = g[0][0] * (g[1][1] * g[2][2] - g[1][2] * g[1][2]) - g[0][1] * (g[0][1] * g[2][2] - g[1][2] * g[0][2]) +
                     g[0][2] * (g[0][1] * g[1][2] - g[1][1] * g[0][2]);
  q.gi[0][0] = (g[1][1] * g[2][2] - g[1][2] * g[1][2]) / det;
  q.gi[0][1] = q.gi[1][0] = (g[0][2] * g[1][2] - g[0][1] * g[2][2]) / det;
  q.gi[0][2] = q.gi[2][0] = (g[0][1] * g[1][2] - g[0][2] * g[1][1]) / det;
  q.gi[1][1] = (g[0][0] * g[2][2] - g[0][2] * g[0][2]) / det;
  q.gi[1][2] = q.gi[2][1] = (g[0][1] * g[0][2] - g[0][0] * g[1][2]) / det;
  q.gi[2][2] = (g[0][0] * g[1][1] - g[0][1] * g[0][1]) / det;
  q.chi = U[(size_t)CHI * n + p];
  q.al = U[(size_t)ALPHA * n + p];
  for (int i = 0; i < 3; ++i) { q.be[i] = U[(size_t)(BETAX + i) * n + p]; q.vu[i] = P[(size_t)(VX + i) * n + p]; }
  for (int a = 0; a < 10; ++a) q.uc[a] = U[(size_t)(DBAR + a) * n + p];
  q.rho = P[(size_t)RHO * n + p]; q.eps = P[(size_t)EPS * n + p]; q.p = P[(size_t)PRESS * n + p];
  q.W = P[(size_t)WLOR * n + p]; q.cs2 = P[(size_t)CS2 * n + p];
}

// densitised stress tensor Sbar_ij = sqrt(gamma) S_ij
static void sbar_ij(const Pt& q, double Sb[3][3]) {
  const double isg = q.chi * std::sqrt(q.chi), sg = 1.0 / isg;
  double gl[3][3], Sl[3], Bu[3], Sij[3][3];
  for (int i = 0; i < 3; ++i) {
    Sl[i] = q.uc[3 + i] * isg; Bu[i] = q.uc[6 + i] * isg;
    for (int j = 0; j < 3; ++j) gl[i][j] = q.g[i][j] / q.chi;
  }
  stress_tensor(gl, q.vu, q.W, q.p, Sl, Bu, Sij);
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Sb[i][j] = sg * Sij[i][j];
}

// flux brackets of Eq. (32) in direction k, and the speed bound s (R12)
static void flux_point(const Params& par, const Pt& q, int k, double F[10], double& s) {
  const double al = q.al, chi = q.chi;
  const double* u = q.uc;   // 0 Dbar 1 DYebar 2 taubar 3-5 Sbar_i 6-8 Bbar^i 9 phibar
  double Sb[3][3];
  sbar_ij(q, Sb);
  const double vk = al * q.vu[k] - q.be[k];               // (-beta^k + alpha v^k)
  F[0] = vk * u[0];
  F[1] = vk * u[1];
  double Sup_k = 0;                                        // Sbar^k = chi gamma~^kj Sbar_j
  for (int j = 0; j < 3; ++j) Sup_k += chi * q.gi[k][j] * u[3 + j];
  F[2] = -q.be[k] * u[2] + al * (Sup_k - u[0] * q.vu[k]);
  for (int i = 0; i < 3; ++i) {
    double Sik = 0;                                        // Sbar_i^k = chi gamma~^kj Sbar_ij
    for (int j = 0; j < 3; ++j) Sik += chi * q.gi[k][j] * Sb[i][j];
    F[3 + i] = -q.be[k] * u[3 + i] + al * Sik;
  }
  for (int i = 0; i < 3; ++i)
    F[6 + i] = u[6 + i] * vk - u[6 + k] * (al * q.vu[i] - q.be[i]) + al * chi * q.gi[k][i] * u[9];
  F[9] = -q.be[k] * u[9] + al * par.c_b * par.c_b * u[6 + k];
  // ---- App. B: fast-magnetosonic bound, Eqs. (B1)-(B3)
  const double isg = chi * std::sqrt(chi);
  double vl[3], Bu[3], Bl[3];
  for (int i = 0; i < 3; ++i) Bu[i] = u[6 + i] * isg;
  for (int i = 0; i < 3; ++i) {
    vl[i] = 0; Bl[i] = 0;
    for (int j = 0; j < 3; ++j) { vl[i] += q.g[i][j] / chi * q.vu[j]; Bl[i] += q.g[i][j] / chi * Bu[j]; }
  }
  double v2 = 0, B2 = 0, Bv = 0;
  for (int i = 0; i < 3; ++i) { v2 += q.vu[i] * vl[i]; B2 += Bu[i] * Bl[i]; Bv += Bu[i] * vl[i]; }
  const double h = q.rho * (1.0 + q.eps) + q.p;            // enthalpy density
  const double b2 = B2 / (q.W * q.W) + Bv * Bv;            // (B3)
  const double ca2 = b2 / (h + b2);
  const double a2 = q.cs2 + ca2 - q.cs2 * ca2;             // (B2)
  const double gkk = chi * q.gi[k][k];                     // gamma^kk
  const double vk_ = q.vu[k];
  const double disc = a2 * (1.0 - v2) * ((1.0 - v2 * a2) * gkk - (1.0 - a2) * vk_ * vk_);
  const double root = std::sqrt(std::max(disc, 0.0));
  const double lp = -q.be[k] + al / (1.0 - v2 * a2) * ((1.0 - a2) * vk_ + root);   // (B1)
  const double lm = -q.be[k] + al / (1.0 - v2 * a2) * ((1.0 - a2) * vk_ - root);
  const double lclean = std::fabs(q.be[k]) + al * par.c_b * std::sqrt(gkk);
  s = std::max(std::max(std::fabs(lp), std::fabs(lm)), lclean);
}

// parts: bit 0 = flux divergence (a6-a7), bit 1 = sources (a8); the split exists only so that the
// operation-counting build can attribute the work to the two steps
void rhs_grmhd_parts(const Params& par, const Grid& G, const double* U, const double* P, double* K, int parts) {
  const size_t n = G.npts();
  const int ng = G.ng;
  const int M[3] = {G.mx(), G.my(), G.mz()};
  const int N[3] = {G.nx, G.ny, G.nz};
  const long st[3] = {1, (long)G.mx(), (long)G.mx() * G.my()};
  const double hh[3] = {G.dx, G.dy, G.dz};
  // zero the interior of the 10 fluid RHS fields
  for (int kk = ng; kk < G.nz + ng; ++kk) for (int jj = ng; jj < G.ny + ng; ++jj) for (int ii = ng; ii < G.nx + ng; ++ii)
    for (int a = 0; a < 10; ++a) K[(size_t)(DBAR + a) * n + G.idx(ii, jj, kk)] = 0.0;

  // ---- LES: the sub-grid-scale tensor of the induction equation is part of the flux bracket of Eq. (32) (App. A; orc_les.cpp)
  std::vector<double> Lsgs, Laux;
  if ((par.les_C_M != 0.0 || par.les_C_N != 0.0 || par.les_C_Y != 0.0 || par.les_C_T != 0.0) && (parts & 1)) {
    Lsgs.resize((size_t)LES_NFLUX * n); Laux.resize((size_t)LES_NAUX * n);
    les_flux(par, G, U, P, Lsgs.data(), Laux.data());
  }
  // ---- flux divergence, direction by direction, line by line (Eqs. 64-69)
  for (int d = 0; d < 3 && (parts & 1); ++d) {
    const int d1_ = (d + 1) % 3, d2_ = (d + 2) % 3;
    const int Md = M[d];
#pragma omp parallel for schedule(dynamic)
    for (int b = ng; b < N[d2_] + ng; ++b) for (int a = ng; a < N[d1_] + ng; ++a) {
      std::vector<double> Fp(10 * Md), Uc(10 * Md), sp(Md), Fhat(10 * (Md + 1));
      int c[3];
      c[d1_] = a; c[d2_] = b; c[d] = 0;
      const size_t base = G.idx(c[0], c[1], c[2]);
      for (int i = 0; i < Md; ++i) {
        Pt q;
        load_point(G, U, P, base + (size_t)i * st[d], q);
        double F[10];
        flux_point(par, q, d, F, sp[i]);
        if (!Lsgs.empty()) {                                          // - alpha G of Eq. (32), direction d
          const size_t q = base + (size_t)i * st[d];
          F[0] += Lsgs[(size_t)(9 + d) * n + q];
          F[1] += Lsgs[(size_t)(12 + d) * n + q];
          for (int c3 = 0; c3 < 3; ++c3) { F[3 + c3] += Lsgs[(size_t)(15 + 3 * d + c3) * n + q]; F[6 + c3] += Lsgs[(size_t)(3 * d + c3) * n + q]; }
        }
        for (int f = 0; f < 10; ++f) { Fp[f * Md + i] = F[f]; Uc[f * Md + i] = q.uc[f]; }
      }
      // interfaces i+1/2 for i = ng-1 .. ng+N-1
      for (int i = ng - 1; i < ng + N[d]; ++i) {
        double lam = 0;                                    // R12: max over the six stencil nodes
        for (int m = i - 2; m <= i + 3; ++m) lam = std::max(lam, sp[m]);
        for (int f = 0; f < 10; ++f) {
          double fpl[6], fmi[6];                           // F^+ and F^- at nodes i-2..i+3, Eq. (65)
          for (int m = 0; m < 6; ++m) {
            const int j = i - 2 + m;
            fpl[m] = 0.5 * (Fp[f * Md + j] + lam * Uc[f * Md + j]);
            fmi[m] = 0.5 * (Fp[f * Md + j] - lam * Uc[f * Md + j]);
          }
          const double FL = reconstruct(par, fpl[0], fpl[1], fpl[2], fpl[3], fpl[4]);   // Eq. (67)
          const double FR = reconstruct(par, fmi[5], fmi[4], fmi[3], fmi[2], fmi[1]);   // Eq. (68)
          Fhat[f * (Md + 1) + i] = FL + FR;                                               // Eq. (69)
        }
      }
      for (int i = ng; i < ng + N[d]; ++i)
        for (int f = 0; f < 10; ++f)
          K[(size_t)(DBAR + f) * n + base + (size_t)i * st[d]] -= (Fhat[f * (Md + 1) + i] - Fhat[f * (Md + 1) + i - 1]) / hh[d];   // Eq. (64)
    }
  }

  // ---- sources of Eq. (32) (+ KO on matter fields if sigma_ko_matter != 0, R16)
  if (parts & 2)
#pragma omp parallel for schedule(dynamic)
  for (int kk = ng; kk < G.nz + ng; ++kk) for (int jj = ng; jj < G.ny + ng; ++jj) for (int ii = ng; ii < G.nx + ng; ++ii) {
    const size_t p = G.idx(ii, jj, kk);
    auto Fd = [&](int f) { return U + (size_t)f * n + p; };
    Pt q;
    load_point(G, U, P, p, q);
    const double al = q.al, chi = q.chi;
    double d_g[3][3][3], d_chi[3], d_al[3], d_be[3][3];
    for (int k = 0; k < 3; ++k) {
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) d_g[k][i][j] = d1(Fd(GXX + SYM[i][j]), st[k], hh[k]);
      d_chi[k] = d1(Fd(CHI), st[k], hh[k]);
      d_al[k] = d1(Fd(ALPHA), st[k], hh[k]);
      for (int i = 0; i < 3; ++i) d_be[k][i] = d1(Fd(BETAX + i), st[k], hh[k]);
    }
    double A[3][3], Gh[3];
    for (int i = 0; i < 3; ++i) { Gh[i] = *Fd(GAMX + i); for (int j = 0; j < 3; ++j) A[i][j] = *Fd(AXX + SYM[i][j]); }
    const double Ktot = *Fd(KHAT) + 2.0 * *Fd(THETA);
    // Z^i = chi/2 (Gamma^^i - Gamma~^i)
    double Z[3];
    for (int k = 0; k < 3; ++k) {
      double Gt = 0;
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int l = 0; l < 3; ++l)
        Gt += q.gi[i][j] * q.gi[k][l] * 0.5 * (d_g[i][l][j] + d_g[j][l][i] - d_g[l][i][j]);
      Z[k] = 0.5 * chi * (Gh[k] - Gt);
    }
    double Sb[3][3], Sbuu[3][3], trS = 0, Sbu[3];
    sbar_ij(q, Sb);
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
      double s = 0;                                        // Sbar^ij = chi^2 gamma~^ik gamma~^jl Sbar_kl
      for (int k = 0; k < 3; ++k) for (int l = 0; l < 3; ++l) s += chi * chi * q.gi[i][k] * q.gi[j][l] * Sb[k][l];
      Sbuu[i][j] = s;
    }
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) trS += q.g[i][j] / chi * Sbuu[i][j];   // tr Sbar = gamma_jk Sbar^jk
    for (int i = 0; i < 3; ++i) { Sbu[i] = 0; for (int j = 0; j < 3; ++j) Sbu[i] += chi * q.gi[i][j] * q.uc[3 + j]; }
    const double* u = q.uc;
    // tau
    double stau = al / 3.0 * trS * Ktot;
    for (int i = 0; i < 3; ++i) {
      stau -= Sbu[i] * d_al[i];
      for (int j = 0; j < 3; ++j) stau += al / chi * Sbuu[i][j] * A[i][j];
    }
    K[(size_t)TAUBAR * n + p] += stau;
    // S_i
    for (int i = 0; i < 3; ++i) {
      double s = -(u[2] + u[0]) * d_al[i] - al / (2.0 * chi) * trS * d_chi[i];
      for (int j = 0; j < 3; ++j) {
        s += u[3 + j] * d_be[i][j];
        for (int k = 0; k < 3; ++k) s += al / (2.0 * chi) * Sbuu[j][k] * d_g[i][j][k];
      }
      K[(size_t)(SXBAR + i) * n + p] += s;
    }
    // B^i
    const double cb2 = par.c_b * par.c_b;
    for (int i = 0; i < 3; ++i) {
      double s = -al * (chi * Gh[i] - 2.0 * Z[i]);
      for (int k = 0; k < 3; ++k) s += q.gi[k][i] * (-0.5 * al * d_chi[k] + chi / cb2 * d_al[k]);
      K[(size_t)(BXBAR + i) * n + p] += u[9] * s;
    }
    // phi
    double sphi = -al * cb2 * u[9] * Ktot - al * par.kappa_b * u[9];
    for (int k = 0; k < 3; ++k) sphi += cb2 * u[6 + k] * d_al[k];
    K[(size_t)PHIBAR * n + p] += sphi;
    if (par.sigma_ko_matter != 0.0)
      for (int a = 0; a < 10; ++a)
        for (int k = 0; k < 3; ++k) K[(size_t)(DBAR + a) * n + p] += dko(Fd(DBAR + a), st[k], hh[k], par.sigma_ko_matter);
  }
}

void rhs_grmhd(const Params& par, const Grid& G, const double* U, const double* P, double* K) {
  rhs_grmhd_parts(par, G, U, P, K, 3);
}

void rhs(const Params& par, const Grid& g, const double* U, const double* P, double* K) {
  rhs_ccz4(par, g, U, P, K);
  rhs_grmhd(par, g, U, P, K);
}

}  // namespace orc
