// ORACLE (test infrastructure) — grey M1 neutrino transport: Minerbo closure (Sec. II C, Eqs. 42-50),
// characteristic speeds (App. B, Eqs. B4-B5), flux-limited advection-diffusion fluxes (Sec. III D, Eqs. 77-78),
// geometric sources of Eqs. (39)-(40), pointwise implicit stiff solve (App. C, Eqs. C10-C35) and the IMEX stage driver
// (Eq. 53, App. C steps C3-C4). Readings R19-R24 of DESIGN.md.
// PARITY UNPINNED: the implicit tableau values (R1) only; see orc.hpp for the list of pins.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>
#include "orc.hpp"

namespace orc {

namespace {
const int SYM_M1[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};

double dot_ud(const double a_up[3], const double b_dn[3]) { return a_up[0] * b_dn[0] + a_up[1] * b_dn[1] + a_up[2] * b_dn[2]; }
void raise(const double gu[3][3], const double a[3], double o[3]) {
  for (int i = 0; i < 3; ++i) o[i] = gu[i][0] * a[0] + gu[i][1] * a[1] + gu[i][2] * a[2];
}
void lower(const double gl[3][3], const double a[3], double o[3]) {
  for (int i = 0; i < 3; ++i) o[i] = gl[i][0] * a[0] + gl[i][1] * a[1] + gl[i][2] * a[2];
}

// J, H.n, H_i and P_ij for a given Eddington factor chi, Eqs. (42)-(48)
void moments_for_chi(double chi, double E, const double F[3], const double Fu[3], double F2, const double vu[3], const double vl[3],
                     double W, const double gl[3][3], M1Closure& c) {
  const double dthin = 0.5 * (3.0 * chi - 1.0), dthick = 1.5 * (1.0 - chi);   // Eq. (48)
  const double W2 = W * W;
  const double Fv = dot_ud(vu, F);
  const double Jthick = 3.0 / (2.0 * W2 + 1.0) * ((2.0 * W2 - 1.0) * E - 2.0 * W2 * Fv);                 // Eq. (47)
  double Hthick_u[3], Hthick[3];
  for (int i = 0; i < 3; ++i)
    Hthick_u[i] = Fu[i] / W + W * vu[i] / (2.0 * W2 + 1.0) * ((4.0 * W2 + 1.0) * Fv - 4.0 * W2 * E);     // l.346
  lower(gl, Hthick_u, Hthick);
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
    const double thin = F2 > 0.0 ? E * F[i] * F[j] / F2 : 0.0;                                           // Eq. (45), R22
    const double thick = 4.0 / 3.0 * Jthick * W2 * vl[i] * vl[j] + W * (Hthick[i] * vl[j] + Hthick[j] * vl[i])
                         + Jthick * gl[i][j] / 3.0;                                                       // Eq. (46)
    c.P[i][j] = dthin * thin + dthick * thick;
  }
  double Pvv = 0.0, Pv[3] = {0, 0, 0};
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { Pvv += c.P[i][j] * vu[i] * vu[j]; Pv[i] += c.P[i][j] * vu[j]; }
  c.J = W2 * (E - 2.0 * Fv + Pvv);                                                                        // Eq. (42)
  c.Hn = W * (c.J - E + Fv);                                                                              // Eq. (43)
  for (int i = 0; i < 3; ++i) c.H[i] = W * (F[i] - Pv[i] - c.J * vl[i]);                                  // Eq. (44)
  c.chi = chi;
}
double eddington(double xi) { return 1.0 / 3.0 + xi * xi * (6.0 - 2.0 * xi + 6.0 * xi * xi) / 15.0; }    // Eq. (49)
}  // namespace

M1Closure m1_closure_point(double E, const double F[3], const double vu[3], double W, const double gl[3][3], const double gu[3][3]) {
  M1Closure c;
  c.fix = 0;
  double Fu[3], vl[3];
  raise(gu, F, Fu);
  lower(gl, vu, vl);
  double F2 = dot_ud(Fu, F);
  if (F2 < 1e-30 * E * E) F2 = 0.0;                                                                       // R22: f^ = 0 for |F| < 1e-15 E
  auto R = [&](double xi) {                                                                               // Eq. (50)
    moments_for_chi(eddington(xi), E, F, Fu, F2, vu, vl, W, gl, c);
    double Hu[3];
    raise(gu, c.H, Hu);
    const double H2 = -c.Hn * c.Hn + dot_ud(Hu, c.H);                                                     // H_a H^a
    return (xi * xi * c.J * c.J - H2) / (E * E);
  };
  double a = 0.0, b = 1.0;
  const double Ra = R(a);
  if (Ra >= 0.0) { c.xi = 0.0; R(0.0); return c; }                  // H = 0: isotropic in the fluid frame
  const double Rb = R(b);
  if (Rb <= 0.0) { c.xi = 1.0; return c; }                          // free streaming (or beyond: |H| >= J)
  // R(0) < 0 < R(1): plain bisection down to neighbouring doubles
  for (int it = 0; it < 200; ++it) {
    const double m = 0.5 * (a + b);
    if (m <= a || m >= b) break;
    const double Rm = R(m);
    if (Rm == 0.0) { a = b = m; break; }
    if (Rm < 0.0) a = m; else b = m;
  }
  c.xi = 0.5 * (a + b);
  R(c.xi);
  return c;
}

// App. C, Eqs. (C17)-(C27)
void m1_JH_appC(double E, const double F[3], const double vu[3], double W, const double gl[3][3], const double gu[3][3],
                double dthin, double dthick, double& J, double H[3]) {
  double Fu[3], vl[3];
  raise(gu, F, Fu);
  lower(gl, vu, vl);
  const double W2 = W * W, v2 = dot_ud(vu, vl), vF = dot_ud(vu, F);
  double F2 = dot_ud(Fu, F);
  double fh[3] = {0, 0, 0};
  if (F2 >= 1e-30 * E * E) { const double Fn = std::sqrt(F2); for (int i = 0; i < 3; ++i) fh[i] = F[i] / Fn; }
  const double vf = dot_ud(vu, fh);
  const double B0 = W2 * (E - 2.0 * vF);                                                                  // (C19)
  const double Bthin = W2 * E * vf * vf;                                                                  // (C20)
  const double Bthick = (W2 - 1.0) / (2.0 * W2 + 1.0) * (4.0 * W2 * vF + (3.0 - 2.0 * W2) * E);           // (C21)
  const double av0 = W * B0, avthin = W * Bthin;                                                          // (C22), (C23)
  const double avthick = W * Bthick + W / (2.0 * W2 + 1.0) * ((2.0 * W2 - 1.0) * vF + (3.0 - 2.0 * W2) * E);   // (C24)
  const double afthin = W * E * vf, aF0 = -W, aFthick = W * v2;                                           // (C25)-(C27)
  J = B0 + dthin * Bthin + dthick * Bthick;                                                               // (C17)
  for (int i = 0; i < 3; ++i)
    H[i] = -(av0 + dthin * avthin + dthick * avthick) * vl[i] - dthin * afthin * fh[i] - (aF0 + dthick * aFthick) * F[i];   // (C18)
}

// Eqs. (C28)-(C35): Jacobian of R_V = alpha (S_n, S_i) with respect to (E, F_j), closure frozen (R21)
void m1_jacobian(double E, const double F[3], const double vu[3], double W, const double gl[3][3], const double gu[3][3],
                 double dthin, double dthick, double alpha, double ka, double ks, double Jac[4][4]) {
  double Fu[3], vl[3];
  raise(gu, F, Fu);
  lower(gl, vu, vl);
  const double W2 = W * W, W3 = W2 * W, v2 = dot_ud(vu, vl), kas = ka + ks;
  double F2 = dot_ud(Fu, F);
  double fh[3] = {0, 0, 0}, fhu[3] = {0, 0, 0}, iF = 0.0;
  if (F2 >= 1e-30 * E * E) { const double Fn = std::sqrt(F2); iF = 1.0 / Fn; for (int i = 0; i < 3; ++i) { fh[i] = F[i] / Fn; fhu[i] = Fu[i] / Fn; } }
  const double vf = dot_ud(vu, fh);
  const double dJdE = W2 + dthin * vf * vf * W2 + dthick * (3.0 - 2.0 * W2) * (W2 - 1.0) / (1.0 + 2.0 * W2);        // (C32)
  double dJdF[3], dHdE[3], dHdF[3][3];
  for (int j = 0; j < 3; ++j)
    dJdF[j] = 2.0 * W2 * (-1.0 + dthin * E * vf * iF + 2.0 * dthick * (W2 - 1.0) / (1.0 + 2.0 * W2)) * vu[j]
              - 2.0 * dthin * W2 * E * vf * vf * iF * fhu[j];                                                         // (C33)
  for (int i = 0; i < 3; ++i)
    dHdE[i] = W3 * (-1.0 - dthin * vf * vf + dthick * (2.0 * W2 - 3.0) / (1.0 + 2.0 * W2)) * vl[i] - dthin * W * vf * fh[i];   // (C34)
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j)
    dHdF[i][j] = W * (1.0 - dthin * E * vf * iF - dthick * v2) * (i == j ? 1.0 : 0.0)
                 + 2.0 * W3 * (1.0 - dthin * E * vf * iF - dthick * (v2 + 1.0 / (2.0 * W2 * (1.0 + 2.0 * W2)))) * vl[i] * vu[j]
                 + 2.0 * dthin * W * E * vf * iF * fh[i] * fhu[j] + 2.0 * dthin * W3 * E * vf * vf * iF * vl[i] * fhu[j]
                 - dthin * W * E * iF * fh[i] * vu[j];                                                                 // (C35)
  Jac[0][0] = -alpha * W * (kas - ks * dJdE);                                                                          // (C28)
  for (int j = 0; j < 3; ++j) Jac[0][1 + j] = alpha * W * (ks * dJdF[j] + kas * vu[j]);                                // (C29)
  for (int i = 0; i < 3; ++i) {
    Jac[1 + i][0] = -alpha * (kas * dHdE[i] + W * ka * dJdE * vl[i]);                                                  // (C30)
    for (int j = 0; j < 3; ++j) Jac[1 + i][1 + j] = -alpha * (kas * dHdF[i][j] + W * ka * vl[i] * dJdF[j]);           // (C31), R23
  }
}

void m1_opacities(const Params& par, int species, double rho, double T, double& ka, double& ks, double& eta) {
  const double x = rho / par.m1_rho0;
  ka = par.m1_kappa0 * x * x * par.m1_species_scale[species];
  ks = ka;
  eta = par.m1_arad * ka * T * T * T * T;
}

namespace {
// R22: floor E, limit |F| <= E; returns true if anything changed
bool m1_fixup(const Params& par, double& E, double F[3], const double gu[3][3]) {
  bool ch = false;
  if (!(E >= par.m1_efloor)) { E = par.m1_efloor; ch = true; }
  double Fu[3];
  raise(gu, F, Fu);
  const double F2 = dot_ud(Fu, F);
  if (F2 > E * E) { const double s = E / std::sqrt(F2); for (int i = 0; i < 3; ++i) F[i] *= s; ch = true; }
  return ch;
}
// alpha (S_n, S_i) of l.312-316 with J, H_i from (C17)-(C18)
void stiff_terms(double E, const double F[3], const double vu[3], double W, const double gl[3][3], const double gu[3][3],
                 double dthin, double dthick, double alpha, double ka, double ks, double eta, double S[4], double& J) {
  double H[3], vl[3];
  m1_JH_appC(E, F, vu, W, gl, gu, dthin, dthick, J, H);
  lower(gl, vu, vl);
  const double Fv = dot_ud(vu, F);
  S[0] = alpha * W * ((eta + ks * J) - (ka + ks) * (E - Fv));
  for (int i = 0; i < 3; ++i) S[1 + i] = alpha * (W * (eta - ka * J) * vl[i] - (ka + ks) * H[i]);
}
bool solve4(double A[4][4], double b[4]) {   // Gaussian elimination with partial pivoting, in place; solution in b
  for (int c = 0; c < 4; ++c) {
    int p = c;
    for (int r = c + 1; r < 4; ++r) if (std::fabs(A[r][c]) > std::fabs(A[p][c])) p = r;
    if (A[p][c] == 0.0) return false;
    if (p != c) { for (int k = 0; k < 4; ++k) std::swap(A[p][k], A[c][k]); std::swap(b[p], b[c]); }
    for (int r = c + 1; r < 4; ++r) {
      const double f = A[r][c] / A[c][c];
      for (int k = c; k < 4; ++k) A[r][k] -= f * A[c][k];
      b[r] -= f * b[c];
    }
  }
  for (int r = 3; r >= 0; --r) {
    double s = b[r];
    for (int k = r + 1; k < 4; ++k) s -= A[r][k] * b[k];
    b[r] = s / A[r][r];
  }
  return true;
}
}  // namespace

uint8_t m1_implicit_point(const Params& par, int species, const double Vstar[5], double adt, double alpha, const double vu[3], double W,
                          double rho, double T, const double gl[3][3], const double gu[3][3], double V[5], double R[5]) {
  uint8_t flag = 0;
  double ka, ks, eta;
  m1_opacities(par, species, rho, T, ka, ks, eta);                  // held fixed during the solve
  double Es = Vstar[1], Fs[3] = {Vstar[2], Vstar[3], Vstar[4]};
  if (m1_fixup(par, Es, Fs, gu)) flag |= FLAG_M1FIX;
  const M1Closure c = m1_closure_point(Es, Fs, vu, W, gl, gu);      // R21: Eddington factor from V*, frozen
  const double dthin = 0.5 * (3.0 * c.chi - 1.0), dthick = 1.5 * (1.0 - c.chi);
  double E = Es, F[3] = {Fs[0], Fs[1], Fs[2]}, J = 0.0, S[4];
  bool conv = adt == 0.0;
  for (int it = 0; it < par.m1_maxit && !conv; ++it) {
    stiff_terms(E, F, vu, W, gl, gu, dthin, dthick, alpha, ka, ks, eta, S, J);
    double G[4] = {E - Es - adt * S[0], F[0] - Fs[0] - adt * S[1], F[1] - Fs[1] - adt * S[2], F[2] - Fs[2] - adt * S[3]};   // (C13)-(C14)
    const double gn = std::max(std::max(std::fabs(G[0]), std::fabs(G[1])), std::max(std::fabs(G[2]), std::fabs(G[3])));
    // R21: the residual is measured against the size of the terms it is made of: E* and the stiff terms a_ii dt alpha W (eta, kappa_as E),
    // whose rounding error bounds what Newton can reach when kappa dt >> 1
    if (gn <= par.m1_tol * (std::max(Es, par.m1_efloor) + adt * alpha * W * (eta + (ka + ks) * std::max(Es, E)))) { conv = true; break; }
    double Jac[4][4], M[4][4];
    m1_jacobian(E, F, vu, W, gl, gu, dthin, dthick, alpha, ka, ks, Jac);
    for (int r = 0; r < 4; ++r) for (int q = 0; q < 4; ++q) M[r][q] = (r == q ? 1.0 : 0.0) - adt * Jac[r][q];               // (C16)
    if (!solve4(M, G)) break;
    E -= G[0]; F[0] -= G[1]; F[1] -= G[2]; F[2] -= G[3];                                                                   // (C15)
  }
  if (!conv) flag |= FLAG_NOCONV;
  if (m1_fixup(par, E, F, gu)) flag |= FLAG_M1FIX;
  stiff_terms(E, F, vu, W, gl, gu, dthin, dthick, alpha, ka, ks, eta, S, J);
  const double Fv = dot_ud(vu, F);
  const double Gam = W * (E - Fv) / J;                                                                                     // (C12)
  const double ka0 = ka, eta0 = eta;                                // synthetic number opacities
  const double N = (Vstar[0] + adt * alpha * eta0) / (1.0 + adt * alpha * ka0 / Gam);                                      // (C11)
  V[0] = N; V[1] = E; V[2] = F[0]; V[3] = F[1]; V[4] = F[2];
  R[0] = alpha * (eta0 - ka0 * N / Gam);                                                                                   // Eq. (41)
  for (int q = 0; q < 4; ++q) R[1 + q] = S[q];
  return flag;
}

}  // namespace orc
