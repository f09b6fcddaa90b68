// ORACLE (test infrastructure) — M1 on a patch: explicit part of Eqs. (38)-(40) with the fluxes of Sec. III D
// (Eqs. 77-78, readings R19, R20), pointwise implicit solve over the patch, fluid back-reaction, IMEX driver (Eq. 53, App. C).
#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>
#include "orc.hpp"

namespace orc {

namespace {
const int SYMP[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};

struct GeoPt {   // geometry and fluid state at one grid point
  double al, be[3], chi, sg, gt[3][3], gl[3][3], gu[3][3];
  double vu[3], W, rho, T;
};
void load_geo(const Grid& G, const double* U, const double* P, size_t p, GeoPt& q) {
  const size_t n = G.npts();
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) q.gt[i][j] = U[(size_t)(GXX + SYMP[i][j]) * n + p];
  const double (*g)[3] = q.gt;
  const double det = g[0][0] * (g[1][1] * g[2][2] - g[1][2] * g[1][2]) - g[0][1] * (g[0][1] * g[2][2] - g[1][2] * g[0][2]) +
                     g[0][2] * (g[0][1] * g[1][2] - g[1][1] * g[0][2]);
  double gi[3][3];
  gi[0][0] = (g[1][1] * g[2][2] - g[1][2] * g[1][2]) / det;
  gi[0][1] = gi[1][0] = (g[0][2] * g[1][2] - g[0][1] * g[2][2]) / det;
  gi[0][2] = gi[2][0] = (g[0][1] * g[1][2] - g[0][2] * g[1][1]) / det;
  gi[1][1] = (g[0][0] * g[2][2] - g[0][2] * g[0][2]) / det;
  gi[1][2] = gi[2][1] = (g[0][1] * g[0][2] - g[0][0] * g[1][2]) / det;
  gi[2][2] = (g[0][0] * g[1][1] - g[0][1] * g[0][1]) / det;
  q.chi = U[(size_t)CHI * n + p];
  q.sg = 1.0 / (q.chi * std::sqrt(q.chi));                         // sqrt(gamma) = chi^(-3/2)
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { q.gl[i][j] = q.gt[i][j] / q.chi; q.gu[i][j] = q.chi * gi[i][j]; }
  q.al = U[(size_t)ALPHA * n + p];
  for (int i = 0; i < 3; ++i) { q.be[i] = U[(size_t)(BETAX + i) * n + p]; q.vu[i] = P[(size_t)(VX + i) * n + p]; }
  q.W = P[(size_t)WLOR * n + p]; q.rho = P[(size_t)RHO * n + p]; q.T = P[(size_t)TEMP * n + p];
}

// pointwise flux brackets of Eqs. (38)-(40) in direction d for one species, state u = (Nbar, Ebar, Fbar_i), speed (B4)-(B5)
void m1_flux_point(const GeoPt& q, const double u[5], int d, double F[5], double& lam) {
  const double E = u[1] / q.sg, Fl[3] = {u[2] / q.sg, u[3] / q.sg, u[4] / q.sg};
  const M1Closure c = m1_closure_point(E, Fl, q.vu, q.W, q.gl, q.gu);
  double Fu[3], Hu[3];
  for (int i = 0; i < 3; ++i) {
    Fu[i] = q.gu[i][0] * Fl[0] + q.gu[i][1] * Fl[1] + q.gu[i][2] * Fl[2];
    Hu[i] = q.gu[i][0] * c.H[0] + q.gu[i][1] * c.H[1] + q.gu[i][2] * c.H[2] + c.Hn * q.be[i] / q.al;   // H^i from l.326
  }
  const double Fv = q.vu[0] * Fl[0] + q.vu[1] * Fl[1] + q.vu[2] * Fl[2];
  const double Gam = q.W * (E - Fv) / c.J;                                                              // l.310
  F[0] = (-q.W * q.be[d] + q.al * q.W * q.vu[d] + q.al * Hu[d] / c.J) * u[0] / Gam;                     // Eq. (38)
  F[1] = -q.be[d] * u[1] + q.al * q.sg * Fu[d];                                                         // Eq. (39)
  for (int i = 0; i < 3; ++i) {
    double Pid = 0.0;                                                                                   // P_i^d
    for (int j = 0; j < 3; ++j) Pid += q.gu[d][j] * c.P[i][j];
    F[2 + i] = -q.be[d] * u[2 + i] + q.al * q.sg * Pid;                                                 // Eq. (40)
  }
  const double F2 = Fu[0] * Fl[0] + Fu[1] * Fl[1] + Fu[2] * Fl[2];
  const double W2 = q.W * q.W;
  double thin = std::fabs(q.be[d]);
  // (B5); R32: the second candidate E |F^d| / F_k F^k equals the first when |F| = E (free streaming) but diverges for
  // |F| << E, where d_thin does not vanish if the fluid moves; no signal outruns light, so the bracket is capped at
  // the coordinate light speed sqrt(gamma^dd)
  if (F2 >= 1e-30 * E * E) thin += q.al * std::min(std::max(std::fabs(Fu[d]) / std::sqrt(F2), E * std::fabs(Fu[d]) / F2), std::sqrt(q.gu[d][d]));
  const double thick = std::fabs(q.be[d]) + q.al * std::max((2.0 * W2 * std::fabs(q.vu[d]) + std::sqrt(std::max((2.0 * W2 + 1.0) * q.gu[d][d] - 2.0 * W2 * q.vu[d] * q.vu[d], 0.0))) / (2.0 * W2 + 1.0),
                                                           std::fabs(q.vu[d]));                       // (B5)
  lam = 0.5 * (3.0 * c.chi - 1.0) * thin + 1.5 * (1.0 - c.chi) * thick;                                 // (B4)
}
}  // namespace

// a11: KV = -div(F^) + geometric sources, interior points; the stiff sources are NOT included
void m1_rhs(const Params& par, const Grid& G, const double* U, const double* P, const double* V, double* KV) {
  const size_t n = G.npts();
  const int ng = G.ng;
  const int M[3] = {G.mx(), G.my(), G.mz()}, N[3] = {G.nx, G.ny, G.nz};
  const long st[3] = {1, (long)G.mx(), (long)G.mx() * G.my()};
  const double hh[3] = {G.dx, G.dy, G.dz};
  for (int f = 0; f < NM1; ++f)
    for (int kk = ng; kk < G.nz + ng; ++kk) for (int jj = ng; jj < G.ny + ng; ++jj) for (int ii = ng; ii < G.nx + ng; ++ii)
      KV[(size_t)f * n + G.idx(ii, jj, kk)] = 0.0;
  for (int s = 0; s < NSPECIES; ++s) for (int d = 0; d < 3; ++d) {
    const int d1_ = (d + 1) % 3, d2_ = (d + 2) % 3, Md = M[d];
#pragma omp parallel for schedule(dynamic)
    for (int b = ng; b < N[d2_] + ng; ++b) for (int a = ng; a < N[d1_] + ng; ++a) {
      std::vector<double> Fp(5 * Md), Uc(5 * Md), lam(Md), kap(Md), Fhat(5 * (Md + 1));
      int c[3];
      c[d1_] = a; c[d2_] = b; c[d] = 0;
      const size_t base = G.idx(c[0], c[1], c[2]);
      for (int i = ng - 2; i < ng + N[d] + 2; ++i) {
        const size_t p = base + (size_t)i * st[d];
        GeoPt q;
        load_geo(G, U, P, p, q);
        double u[5], F[5];
        for (int f = 0; f < 5; ++f) u[f] = V[(size_t)(5 * s + f) * n + p];
        m1_flux_point(q, u, d, F, lam[i]);
        double ka, ks, eta;
        m1_opacities(par, s, q.rho, q.T, ka, ks, eta);
        kap[i] = ka + ks;
        for (int f = 0; f < 5; ++f) { Fp[f * Md + i] = F[f]; Uc[f * Md + i] = u[f]; }
      }
      for (int i = ng - 1; i < ng + N[d]; ++i) {                    // interface i + 1/2
        const double l = std::max(lam[i], lam[i + 1]);
        const double kh = 0.5 * (kap[i] + kap[i + 1]);              // l.561
        const double A0 = kh * hh[d] > 0.0 ? std::tanh(1.0 / (kh * hh[d])) : 1.0;
        for (int f = 0; f < 5; ++f) {
          const double* u = &Uc[f * Md];
          const double* F = &Fp[f * Md];
          const double dm = u[i] - u[i - 1], d0 = u[i + 1] - u[i], dp = u[i + 2] - u[i + 1];
          const double Phi = d0 == 0.0 ? 1.0 : std::max(0.0, std::min(1.0, std::min(2.0 * dm / d0, 2.0 * dp / d0)));   // Eq. (78), R20
          double A = A0;
          // odd-even decoupling, l.565-570, as printed: A := 1 when (u_i - u_{i-1})(u_{i+1} - u_i) < 0 and
          // (u_{i+1} - u_i)(u_{i+2} - u_{i+1}) < 0. Reading R33 (a DEPARTURE from the printed rule, off when m1_oe_guard = 0):
          // the three differences must also exceed m1_oe_guard x the local magnitude, so that a zigzag of rounding noise on a
          // flat profile does not count as an oscillation
          const double tiny = par.m1_oe_guard * std::max(std::max(std::fabs(u[i - 1]), std::fabs(u[i])), std::max(std::fabs(u[i + 1]), std::fabs(u[i + 2])));
          if (par.m1_odd_even && dm * d0 < 0.0 && d0 * dp < 0.0 && std::min(std::min(std::fabs(dm), std::fabs(d0)), std::fabs(dp)) > tiny) A = 1.0;
          const double FHO = 0.5 * (F[i] + F[i + 1]);
          const double FLO = FHO - 0.5 * l * d0;                    // R20
          Fhat[f * (Md + 1) + i] = FHO - A * (1.0 - Phi) * (FHO - FLO);                                                 // Eq. (77)
        }
      }
      for (int i = ng; i < ng + N[d]; ++i)
        for (int f = 0; f < 5; ++f)
          KV[(size_t)(5 * s + f) * n + base + (size_t)i * st[d]] -= (Fhat[f * (Md + 1) + i] - Fhat[f * (Md + 1) + i - 1]) / hh[d];
    }
  }
  // geometric sources of Eqs. (39)-(40)
#pragma omp parallel for schedule(dynamic)
  for (int kk = ng; kk < G.nz + ng; ++kk) for (int jj = ng; jj < G.ny + ng; ++jj) for (int ii = ng; ii < G.nx + ng; ++ii) {
    const size_t p = G.idx(ii, jj, kk);
    auto Fd = [&](int f) { return U + (size_t)f * n + p; };
    GeoPt q;
    load_geo(G, U, P, p, q);
    double d_g[3][3][3], d_chi[3], d_al[3], d_be[3][3], At[3][3];
    for (int k = 0; k < 3; ++k) {
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) d_g[k][i][j] = d1(Fd(GXX + SYMP[i][j]), st[k], hh[k]);
      d_chi[k] = d1(Fd(CHI), st[k], hh[k]);
      d_al[k] = d1(Fd(ALPHA), st[k], hh[k]);
      for (int i = 0; i < 3; ++i) d_be[k][i] = d1(Fd(BETAX + i), st[k], hh[k]);
    }
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) At[i][j] = *Fd(AXX + SYMP[i][j]);
    const double Ktot = *Fd(KHAT) + 2.0 * *Fd(THETA);
    for (int s = 0; s < NSPECIES; ++s) {
      double u[5];
      for (int f = 0; f < 5; ++f) u[f] = V[(size_t)(5 * s + f) * n + p];
      const double E = u[1] / q.sg, Fl[3] = {u[2] / q.sg, u[3] / q.sg, u[4] / q.sg};
      const M1Closure c = m1_closure_point(E, Fl, q.vu, q.W, q.gl, q.gu);
      double Pbuu[3][3], trP = 0.0, Fbu[3];
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
        double sum = 0.0;
        for (int k = 0; k < 3; ++k) for (int l = 0; l < 3; ++l) sum += q.gu[i][k] * q.gu[j][l] * c.P[k][l];
        Pbuu[i][j] = q.sg * sum;
      }
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) trP += q.gl[i][j] * Pbuu[i][j];
      for (int i = 0; i < 3; ++i) Fbu[i] = q.gu[i][0] * u[2] + q.gu[i][1] * u[3] + q.gu[i][2] * u[4];
      double sE = q.al / 3.0 * trP * Ktot;
      for (int i = 0; i < 3; ++i) {
        sE -= Fbu[i] * d_al[i];
        for (int j = 0; j < 3; ++j) sE += q.al / q.chi * Pbuu[i][j] * At[i][j];                          // R19
      }
      KV[(size_t)(5 * s + 1) * n + p] += sE;
      for (int i = 0; i < 3; ++i) {
        double sF = -u[1] * d_al[i] - q.al / (2.0 * q.chi) * trP * d_chi[i];
        for (int j = 0; j < 3; ++j) {
          sF += u[2 + j] * d_be[i][j];
          for (int k = 0; k < 3; ++k) sF += q.al / (2.0 * q.chi) * Pbuu[j][k] * d_g[i][j][k];
        }
        KV[(size_t)(5 * s + 2 + i) * n + p] += sF;
      }
    }
  }
}

// a12 over the patch (every point incl. ghosts): V holds V* on entry (densitised), V^(i) on exit; R = densitised stiff source
void m1_implicit(const Params& par, const Grid& G, const double* U, const double* P, double* V, double* R, double adt, uint8_t* flags) {
  const size_t n = G.npts();
#pragma omp parallel for schedule(dynamic, 512)
  for (size_t p = 0; p < n; ++p) {
    GeoPt q;
    load_geo(G, U, P, p, q);
    for (int s = 0; s < NSPECIES; ++s) {
      double vs[5], v[5], r[5];
      for (int f = 0; f < 5; ++f) vs[f] = V[(size_t)(5 * s + f) * n + p] / q.sg;
      const uint8_t fl = m1_implicit_point(par, s, vs, adt, q.al, q.vu, q.W, q.rho, q.T, q.gl, q.gu, v, r);
      if (flags) flags[p] |= fl;
      for (int f = 0; f < 5; ++f) { V[(size_t)(5 * s + f) * n + p] = q.sg * v[f]; R[(size_t)(5 * s + f) * n + p] = q.sg * r[f]; }
    }
  }
}

// neutrino back-reaction on the fluid (l.256, l.312-316; R24): K[taubar] -= sum R[Ebar], K[Sbar_i] -= sum R[Fbar_i],
// K[DYebar] -= m_b (R[Nbar]_nue - R[Nbar]_nuebar), with R the stored stiff source of the same stage
void m1_backreaction(const Params& par, const Grid& G, const double* U, const double* P, const double* R, double* K) {
  (void)U; (void)P;
  const size_t n = G.npts();
  const int ng = G.ng;
  for (int kk = ng; kk < G.nz + ng; ++kk) for (int jj = ng; jj < G.ny + ng; ++jj) for (int ii = ng; ii < G.nx + ng; ++ii) {
    const size_t p = G.idx(ii, jj, kk);
    for (int s = 0; s < NSPECIES; ++s) {
      K[(size_t)TAUBAR * n + p] -= R[(size_t)(5 * s + 1) * n + p];
      for (int i = 0; i < 3; ++i) K[(size_t)(SXBAR + i) * n + p] -= R[(size_t)(5 * s + 2 + i) * n + p];
    }
    K[(size_t)DYEBAR * n + p] -= par.m1_mb * (R[(size_t)0 * n + p] - R[(size_t)5 * n + p]);
  }
}

// a4 with M1 on (R6, second half): the radiation energy density, momentum density and stresses of all species are added to
// the matter sources of the CCZ4 equations. They enter Eqs. (14), (16), (17), (19) linearly:
//   d_t K^      += alpha 4 pi G (E + S),            S = gamma^ij P_ij
//   d_t Theta   -= alpha 8 pi G E
//   d_t A~_ij   -= alpha 8 pi G chi [P_ij - gamma~_ij gamma~^kl P_kl / 3]
//   d_t Gamma^^i -= 16 pi G alpha gamma~^ij F_j
void m1_gravity(const Params& par, const Grid& G, const double* U, const double* P, const double* V, double* K) {
  const size_t n = G.npts();
  const int ng = G.ng;
  const double G8 = 8.0 * 3.14159265358979323846 * par.grav_G;
  if (G8 == 0.0) return;
#pragma omp parallel for schedule(dynamic)
  for (int kk = ng; kk < G.nz + ng; ++kk) for (int jj = ng; jj < G.ny + ng; ++jj) for (int ii = ng; ii < G.nx + ng; ++ii) {
    const size_t p = G.idx(ii, jj, kk);
    GeoPt q;
    load_geo(G, U, P, p, q);
    double E = 0.0, F[3] = {0, 0, 0}, Pij[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    for (int s = 0; s < NSPECIES; ++s) {
      const double Es = V[(size_t)(5 * s + 1) * n + p] / q.sg;
      const double Fs[3] = {V[(size_t)(5 * s + 2) * n + p] / q.sg, V[(size_t)(5 * s + 3) * n + p] / q.sg, V[(size_t)(5 * s + 4) * n + p] / q.sg};
      const M1Closure c = m1_closure_point(Es, Fs, q.vu, q.W, q.gl, q.gu);
      E += Es;
      for (int i = 0; i < 3; ++i) { F[i] += Fs[i]; for (int j = 0; j < 3; ++j) Pij[i][j] += c.P[i][j]; }
    }
    double S = 0.0;
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) S += q.gu[i][j] * Pij[i][j];
    K[(size_t)KHAT * n + p] += q.al * 0.5 * G8 * (E + S);
    K[(size_t)THETA * n + p] -= q.al * G8 * E;
    for (int i = 0; i < 3; ++i) for (int j = i; j < 3; ++j)
      K[(size_t)(AXX + SYMP[i][j]) * n + p] -= q.al * G8 * q.chi * (Pij[i][j] - q.gt[i][j] * (S / q.chi) / 3.0);
    for (int i = 0; i < 3; ++i) {
      double Fu = 0.0;                                   // gamma~^ij F_j = gamma^ij F_j / chi
      for (int j = 0; j < 3; ++j) Fu += q.gu[i][j] / q.chi * F[j];
      K[(size_t)(GAMX + i) * n + p] -= 2.0 * q.al * G8 * Fu;
    }
  }
}

void evolve_imex(const Params& par, const Grid& g, double* U, double* V, double* P, uint8_t* flags, const int bc[6], int stages,
                 const double* ae, const double* we, const double* ai, const double* wi, double dt, int n_steps) {
  const size_t nu = (size_t)NSTATE * g.npts(), nv = (size_t)NM1 * g.npts();
  std::vector<double> U0(nu), V0(nv);
  std::vector<std::vector<double>> K(stages, std::vector<double>(nu, 0.0)), KV(stages, std::vector<double>(nv, 0.0)), R(stages, std::vector<double>(nv, 0.0));
  std::vector<const double*> Kp(stages), KVp(stages), Rp(stages);
  for (int s = 0; s < stages; ++s) { Kp[s] = K[s].data(); KVp[s] = KV[s].data(); Rp[s] = R[s].data(); }
  for (int step = 0; step < n_steps; ++step) {
    fill_ghosts(g, U, NSTATE, bc);
    con2prim(par, g, U, P, flags);
    fill_ghosts(g, V, NM1, bc);
    std::memcpy(U0.data(), U, nu * sizeof(double));
    std::memcpy(V0.data(), V, nv * sizeof(double));
    for (int s = 0; s < stages; ++s) {
      if (s > 0) {
        // explicit intermediate values W*, V* (C3)
        rk_combine(g, NSTATE, U, U0.data(), s, Kp.data(), ae + (size_t)s * stages, dt);
        rk_combine(g, NM1, V, V0.data(), s, KVp.data(), ae + (size_t)s * stages, dt);
        rk_combine(g, NM1, V, V, s, Rp.data(), ai + (size_t)s * stages, dt);
        fill_ghosts(g, U, NSTATE, bc);
        con2prim(par, g, U, P, flags);
        fill_ghosts(g, V, NM1, bc);
      }
      m1_implicit(par, g, U, P, V, R[s].data(), ai[(size_t)s * stages + s] * dt, flags);   // (C4)
      rhs(par, g, U, P, K[s].data());
      m1_backreaction(par, g, U, P, R[s].data(), K[s].data());
      m1_gravity(par, g, U, P, V, K[s].data());
      m1_rhs(par, g, U, P, V, KV[s].data());
    }
    rk_combine(g, NSTATE, U, U0.data(), stages, Kp.data(), we, dt);
    rk_combine(g, NM1, V, V0.data(), stages, KVp.data(), we, dt);
    rk_combine(g, NM1, V, V, stages, Rp.data(), wi, dt);
  }
  fill_ghosts(g, U, NSTATE, bc);
  con2prim(par, g, U, P, flags);
  fill_ghosts(g, V, NM1, bc);
}

}  // namespace orc
