// ORACLE (test infrastructure) — conserved <-> primitive, Eq. (29) l.223-232 and
// App. D l.1081-1162 (RePrimAnd-style recovery with two bracketed root solves; the oracle solves both by bisection).
#include <algorithm>
#include <cfloat>
#include <cmath>
#include "orc.hpp"

namespace orc {

static void lower(const double gl[6], const double v[3], double out[3]) {
  out[0] = gl[0] * v[0] + gl[1] * v[1] + gl[2] * v[2];
  out[1] = gl[1] * v[0] + gl[3] * v[1] + gl[4] * v[2];
  out[2] = gl[2] * v[0] + gl[4] * v[1] + gl[5] * v[2];
}
static void inv_sym(const double g[6], double gi[6], double& det) {
  const double xx = g[0], xy = g[1], xz = g[2], yy = g[3], yz = g[4], zz = g[5];
  det = xx * (yy * zz - yz * yz) - xy * (xy * zz - yz * xz) + xz * (xy * yz - yy * xz);
  gi[0] = (yy * zz - yz * yz) / det;
  gi[1] = (xz * yz - xy * zz) / det;
  gi[2] = (xy * yz - xz * yy) / det;
  gi[3] = (xx * zz - xz * xz) / det;
  gi[4] = (xy * xz - xx * yz) / det;
  gi[5] = (xx * yy - xy * xy) / det;
}

// Eq. (29); h = rho(1+eps)+p is the enthalpy density; v^i contravariant in prim
void prim2con_point(const double gl[6], const double prim[NPRIM], const double B[3],
                    double& D, double& tau, double S[3]) {
  const double v[3] = {prim[VX], prim[VY], prim[VZ]};
  double vl[3], Bl[3];
  lower(gl, v, vl);
  lower(gl, B, Bl);
  const double v2 = v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2];
  const double B2 = B[0] * Bl[0] + B[1] * Bl[1] + B[2] * Bl[2];
  const double Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2];
  const double W2 = 1.0 / (1.0 - v2);
  const double W = std::sqrt(W2);
  const double h = prim[RHO] * (1.0 + prim[EPS]) + prim[PRESS];
  D = prim[RHO] * W;
  tau = h * W2 - prim[PRESS] + B2 - 0.5 * (Bv * Bv + B2 / W2) - D;
  for (int i = 0; i < 3; ++i) S[i] = (h * W2 + B2) * vl[i] - Bv * Bl[i];
}

// Root of f on [a, b] with f(a) f(b) <= 0 by plain bisection until the two ends are adjacent doubles (R9: App. D asks for a
// bracketing solver, "Brent" at l.1114, l.1143; the root in the bracket is unique, so every convergent bracketing method
// returns the same number to rounding — the oracle uses the simplest one). The end whose |f| is smaller is returned.
// conv = false if maxit halvings were not enough.
template <class F>
static double bisect_root(F&& f, double a, double b, double fa, double fb, int maxit, bool& conv) {
  conv = true;
  if (fa == 0.0) return a;
  if (fb == 0.0) return b;
  for (int it = 0; it < maxit; ++it) {
    const double m = a + 0.5 * (b - a);
    if (m == a || m == b) return std::fabs(fa) <= std::fabs(fb) ? a : b;
    const double fm = f(m);
    if (fm == 0.0) return m;
    if ((fm > 0.0) == (fa > 0.0)) { a = m; fa = fm; } else { b = m; fb = fm; }
  }
  conv = false;
  return std::fabs(fa) <= std::fabs(fb) ? a : b;
}

namespace {
struct C2P {
  const Params& par;
  double D, q, r2, B2, rB2, B2rperp2, ye, h0, v02, rho_lo, rho_hi;
  // outputs of the last evaluation of f
  double rho, eps, eps_raw, p, W, T, cs2;

  double chi(double mu) const { return 1.0 / (1.0 + mu * B2); }                        // (D5)
  double rbar2(double mu) const {                                                      // (D4)
    const double x = chi(mu);
    return r2 * x * x + mu * x * (1.0 + x) * rB2;
  }
  double fa(double mu) const { return mu * std::sqrt(h0 * h0 + rbar2(mu)) - 1.0; }     // (D3)
  double f(double mu) {                                                                // (D6)
    const double x = chi(mu);
    const double rb2 = rbar2(mu);
    const double qbar = q - 0.5 * B2 - 0.5 * mu * mu * x * x * B2rperp2;               // (D14)
    const double v2 = std::min(mu * mu * rb2, v02);                                    // (D13)
    W = 1.0 / std::sqrt(1.0 - v2);
    rho = D / W;                                                                       // (D11)
    rho = std::max(std::min(rho_hi, rho), rho_lo);                                     // l.1145
    eps_raw = W * (qbar - mu * rb2) + v2 * W * W / (1.0 + W);                          // (D12)
    double emin, emax;
    eos_eps_range(par, rho, ye, emin, emax);
    eps = std::max(std::min(emax, eps_raw), emin);                                     // l.1145
    const EosOut e = eos_from_rho_eps(par, rho, eps, ye);                              // (D10)
    p = e.p; T = e.T; cs2 = e.cs2;
    const double a = p / (rho * (1.0 + eps));
    const double nuA = (1.0 + a) * (1.0 + eps) / W;                                    // (D8)
    const double nuB = (1.0 + a) * (1.0 + qbar - mu * rb2);                            // (D9)
    const double nu = std::max(nuA, nuB);                                              // (D7)
    return mu - 1.0 / (nu + mu * rb2);
  }
};
}  // namespace

// ucons = {Dbar, DYebar, taubar, Sbar_x, Sbar_y, Sbar_z, Bbar^x, Bbar^y, Bbar^z, phibar}
uint8_t con2prim_point(const Params& par, const double gt[6], double chi, double alpha,
                       double uc[10], double prim[NPRIM]) {
  uint8_t flag = 0;
  // undensitise: sqrt(gamma) = chi^(-3/2)  (det gamma~ = 1);  note N2: D = Dbar * (chi * sqrt(chi))
  const double isg = chi * std::sqrt(chi);
  const double sg = 1.0 / isg;
  const double D = uc[0] * isg;
  double gl[6], gti[6], gu[6], det;
  for (int a = 0; a < 6; ++a) gl[a] = gt[a] / chi;         // gamma_ij = gamma~_ij / chi  (l.132)
  inv_sym(gt, gti, det);
  for (int a = 0; a < 6; ++a) gu[a] = chi * gti[a];        // gamma^ij = chi gamma~^ij
  const double B[3] = {uc[6] * isg, uc[7] * isg, uc[8] * isg};
  double ye = uc[1] / uc[0];

  double rho = 0, eps = 0, W = 1, v[3] = {0, 0, 0};
  bool atmo = !(D >= par.rho_cut);                          // rule 1 pre-check (N2); also catches NaN
  bool changed = false;
  const bool bh = alpha < par.alpha_bh;

  if (!atmo) {
    const double tau = uc[2] * isg;
    const double Sl[3] = {uc[3] * isg, uc[4] * isg, uc[5] * isg};
    // (D1)-(D2)
    const double q = tau / D;
    const double rl[3] = {Sl[0] / D, Sl[1] / D, Sl[2] / D};
    const double sD = std::sqrt(D);
    const double Bs[3] = {B[0] / sD, B[1] / sD, B[2] / sD};
    double ru[3], Bsl[3];
    lower(gu, rl, ru);
    lower(gl, Bs, Bsl);
    C2P s{par};
    s.D = D; s.q = q; s.ye = std::max(std::min(ye, par.ye_max), par.ye_min);
    s.r2 = ru[0] * rl[0] + ru[1] * rl[1] + ru[2] * rl[2];
    s.B2 = Bs[0] * Bsl[0] + Bs[1] * Bsl[1] + Bs[2] * Bsl[2];
    const double rB = rl[0] * Bs[0] + rl[1] * Bs[1] + rl[2] * Bs[2];
    s.rB2 = rB * rB;
    s.B2rperp2 = s.B2 * s.r2 - s.rB2;
    s.h0 = eos_h0(par);
    s.v02 = s.r2 / (s.h0 * s.h0 + s.r2);
    eos_rho_range(par, s.rho_lo, s.rho_hi);
    // step 2: root of f_a on (0, 1/h0]
    bool c1 = true, c2 = true;
    const double mub = 1.0 / s.h0;
    const double mu_plus = bisect_root([&](double m) { return s.fa(m); }, 0.0, mub, -1.0, s.fa(mub), std::max(par.c2p_maxit, 1100), c1);
    // step 3: root of f on (0, mu_plus]
    const double f0 = s.f(0.0), f1 = s.f(mu_plus);
    double mu;
    // no sign change: the root sits at the bracket end when the state is degenerate (eps clamped to its minimum gives
    // h = h0 and f(mu_plus) = 0 analytically, +-1e-16 numerically): that is a converged solve, not a failure (R9)
    if ((f0 > 0.0) == (f1 > 0.0) && f1 != 0.0 && f0 != 0.0) { mu = mu_plus; c2 = std::fabs(f1) <= 1e-12; }
    else mu = bisect_root([&](double m) { return s.f(m); }, 0.0, mu_plus, f0, f1, std::max(par.c2p_maxit, 1100), c2);
    s.f(mu);                                                // step 4: primitives at the root
    if (!c1 || !c2) flag |= FLAG_NOCONV;
    rho = D / s.W; W = s.W; eps = s.eps_raw;
    const double x = s.chi(mu);
    for (int i = 0; i < 3; ++i) v[i] = mu * x * (ru[i] + mu * rB * Bs[i]);   // (D15), contravariant
    // ---- error policy
    if (!(rho >= par.rho_cut)) atmo = true;                 // rule 1
    else {
      const bool low = rho < par.rho_low;
      const bool allowed = low || bh;
      if (rho > par.rho_max) flag |= FLAG_FATAL;            // rule 2
      double emin, emax;
      const double rho_c = std::max(std::min(s.rho_hi, rho), s.rho_lo);
      eos_eps_range(par, rho_c, s.ye, emin, emax);
      if (eps < emin) { eps = emin; flag |= FLAG_EPS_LO; changed = true; }          // rule 3
      else if (eps > emax) {                                                        // rule 4
        eps = emax; changed = true;
        flag |= allowed ? FLAG_EPS_HI : (FLAG_EPS_HI | FLAG_FATAL);
      }
      if (W > par.w_max) {                                                          // rule 5
        flag |= allowed ? FLAG_VMAX : (FLAG_VMAX | FLAG_FATAL);
        const double vmax2 = 1.0 - 1.0 / (par.w_max * par.w_max);
        double vl[3];
        lower(gl, v, vl);
        const double v2 = v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2];
        const double sc = std::sqrt(vmax2 / v2);
        for (int i = 0; i < 3; ++i) v[i] *= sc;
        W = par.w_max;
        rho = D / W;                                        // D kept fixed: rho increases slightly
        changed = true;
      }
      if (ye < par.ye_min || ye > par.ye_max) {                                     // rule 6
        flag |= allowed ? FLAG_YE : (FLAG_YE | FLAG_FATAL);
        ye = par.ye_atmo; changed = true;
      }
    }
  }
  if (atmo) {                                               // rule 1: reset to atmosphere
    flag |= FLAG_ATMO;
    rho = par.rho_atmo; W = 1.0; v[0] = v[1] = v[2] = 0.0; ye = par.ye_atmo;
    eps = par.eos_kind == 2 ? eos_eps_from_T(par, rho, par.T_atmo, ye) : par.eps_atmo;
    if (par.eos_kind == 1) { double emin, emax; eos_eps_range(par, rho, ye, emin, emax); eps = emin + par.eps_atmo; }
    changed = true;
  }
  const EosOut e = eos_from_rho_eps(par, rho, eps, ye);
  prim[RHO] = rho; prim[YE] = ye; prim[EPS] = eps; prim[PRESS] = e.p;
  prim[VX] = v[0]; prim[VY] = v[1]; prim[VZ] = v[2]; prim[WLOR] = W; prim[TEMP] = e.T; prim[CS2] = e.cs2;
  if (changed) {                                            // R11: conserved reset from corrected primitives
    double Dn, taun, Sn[3];
    prim2con_point(gl, prim, B, Dn, taun, Sn);
    uc[0] = sg * Dn; uc[1] = sg * Dn * ye; uc[2] = sg * taun;
    uc[3] = sg * Sn[0]; uc[4] = sg * Sn[1]; uc[5] = sg * Sn[2];
  }
  return flag;
}

void con2prim(const Params& par, const Grid& g, double* U, double* P, uint8_t* flags) {
  const size_t n = g.npts();
#pragma omp parallel for schedule(dynamic, 512)
  for (size_t p = 0; p < n; ++p) {
    double gt[6], uc[10], prim[NPRIM];
    for (int a = 0; a < 6; ++a) gt[a] = U[(GXX + a) * n + p];
    for (int a = 0; a < 10; ++a) uc[a] = U[(DBAR + a) * n + p];
    flags[p] = con2prim_point(par, gt, U[CHI * n + p], U[ALPHA * n + p], uc, prim);
    for (int a = 0; a < 10; ++a) U[(DBAR + a) * n + p] = uc[a];
    for (int a = 0; a < NPRIM; ++a) P[a * n + p] = prim[a];
  }
}

// patch-level prim -> conserved: P holds rho, Ye, eps, v^i on entry; p, W, T, cs2 are filled from the EoS
// and the densitised Dbar, DYebar, taubar, Sbar_i are written into U (Bbar^i, phibar and the metric are inputs).
void prim2con(const Params& par, const Grid& g, double* U, double* P) {
  const size_t n = g.npts();
#pragma omp parallel for schedule(dynamic, 512)
  for (size_t p = 0; p < n; ++p) {
    const double chi = U[CHI * n + p];
    const double isg = chi * std::sqrt(chi), sg = 1.0 / isg;
    double gl[6], prim[NPRIM], D, tau, S[3];
    for (int a = 0; a < 6; ++a) gl[a] = U[(GXX + a) * n + p] / chi;
    for (int a = 0; a < NPRIM; ++a) prim[a] = P[a * n + p];
    const EosOut e = eos_from_rho_eps(par, prim[RHO], prim[EPS], prim[YE]);
    prim[PRESS] = e.p; prim[TEMP] = e.T; prim[CS2] = e.cs2;
    const double B[3] = {U[BXBAR * n + p] * isg, U[BYBAR * n + p] * isg, U[BZBAR * n + p] * isg};
    prim2con_point(gl, prim, B, D, tau, S);
    const double v[3] = {prim[VX], prim[VY], prim[VZ]};
    double vl[3];
    lower(gl, v, vl);
    prim[WLOR] = 1.0 / std::sqrt(1.0 - (v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2]));
    for (int a = 0; a < NPRIM; ++a) P[a * n + p] = prim[a];
    U[DBAR * n + p] = sg * D; U[DYEBAR * n + p] = sg * D * prim[YE]; U[TAUBAR * n + p] = sg * tau;
    U[SXBAR * n + p] = sg * S[0]; U[SYBAR * n + p] = sg * S[1]; U[SZBAR * n + p] = sg * S[2];
  }
}

}  // namespace orc
