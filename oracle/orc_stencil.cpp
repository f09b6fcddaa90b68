// ORACLE (test infrastructure) — finite-difference stencils and MP5, Sec. III B-C.
// All zero-sum stencils are evaluated on differences from the centre (DESIGN.md note N1):
// algebraically identical to the printed coefficients, but free of cancellation noise.
#include <algorithm>
#include <cmath>
#include "orc.hpp"

namespace orc {

// Eq. (60):  (U[-2] - 8 U[-1] + 8 U[+1] - U[+2]) / (12 h)
double d1(const double* u, long s, double h) {
  return (8.0 * (u[s] - u[-s]) - (u[2 * s] - u[-2 * s])) / (12.0 * h);
}

// Eq. (62):  (-U[-2] + 16 U[-1] - 30 U[0] + 16 U[+1] - U[+2]) / (12 h^2)
double d2(const double* u, long s, double h) {
  const double u0 = u[0];
  return (16.0 * ((u[s] - u0) + (u[-s] - u0)) - ((u[2 * s] - u0) + (u[-2 * s] - u0))) / (12.0 * h * h);
}

// Eq. (61):  D_y (D_x U)
double d11(const double* u, long s1, double h1, long s2, double h2) {
  const double a = d1(u + s2, s1, h1), b = d1(u - s2, s1, h1);
  const double c = d1(u + 2 * s2, s1, h1), d = d1(u - 2 * s2, s1, h1);
  return (8.0 * (a - b) - (c - d)) / (12.0 * h2);
}

// One-sided advective derivative, PAPER.md:454-456 (R15: beta >= 0 takes the "beta > 0" branch)
//  beta<0: (-U[-3] + 6 U[-2] - 18 U[-1] + 10 U[0] + 3 U[+1]) / (12 h)
//  beta>0: ( U[+3] - 6 U[+2] + 18 U[+1] - 10 U[0] - 3 U[-1]) / (12 h)
double dadv(const double* u, long s, double h, double beta) {
  const double u0 = u[0];
  if (beta < 0.0)
    return (-(u[-3 * s] - u0) + 6.0 * (u[-2 * s] - u0) - 18.0 * (u[-s] - u0) + 3.0 * (u[s] - u0)) / (12.0 * h);
  return ((u[3 * s] - u0) - 6.0 * (u[2 * s] - u0) + 18.0 * (u[s] - u0) - 3.0 * (u[-s] - u0)) / (12.0 * h);
}

// Kreiss-Oliger: sigma/(64 h) (U[-3] - 6U[-2] + 15U[-1] - 20U[0] + 15U[+1] - 6U[+2] + U[+3])
double dko(const double* u, long s, double h, double sigma) {
  const double u0 = u[0];
  return sigma / (64.0 * h) *
         (((u[-3 * s] - u0) + (u[3 * s] - u0)) - 6.0 * ((u[-2 * s] - u0) + (u[2 * s] - u0)) +
          15.0 * ((u[-s] - u0) + (u[s] - u0)));
}

// Minmod of two and four arguments, PAPER.md:516 (R14: common sign x smallest magnitude, else 0)
static double minmod2(double a, double b) {
  const double sa = (a > 0.0) - (a < 0.0), sb = (b > 0.0) - (b < 0.0);
  return 0.5 * (sa + sb) * std::min(std::fabs(a), std::fabs(b));
}
static double minmod4(double a, double b, double c, double d) {
  if (a > 0.0 && b > 0.0 && c > 0.0 && d > 0.0) return std::min(std::min(a, b), std::min(c, d));
  if (a < 0.0 && b < 0.0 && c < 0.0 && d < 0.0) return std::max(std::max(a, b), std::max(c, d));
  return 0.0;
}
static double median3(double a, double b, double c) { return a + minmod2(b - a, c - a); }

// R_MP5(F_{i-2}, F_{i-1}, F_i, F_{i+1}, F_{i+2}), Eqs. (70)-(76)
double mp5(double fm2, double fm1, double f0, double fp1, double fp2, double alpha) {
  const double fhi = (2.0 * fm2 - 13.0 * fm1 + 47.0 * f0 + 27.0 * fp1 - 3.0 * fp2) / 60.0;  // Eq. (70)
  const double dmh = f0 - fm1;   // Delta_{i-1/2}
  const double dph = fp1 - f0;   // Delta_{i+1/2}
  const double fmp = f0 + minmod2(dph, alpha * dmh);                                        // Eq. (71)
  if ((fhi - f0) * (fhi - fmp) < 0.0) return fhi;                                           // Eq. (72)
  const double dm1 = fm2 - 2.0 * fm1 + f0;   // d_{i-1}
  const double d0 = fm1 - 2.0 * f0 + fp1;    // d_i
  const double dp1 = f0 - 2.0 * fp1 + fp2;   // d_{i+1}
  const double dm4_ph = minmod4(4.0 * d0 - dp1, 4.0 * dp1 - d0, d0, dp1);                   // Eq. (76), i+1/2
  const double dm4_mh = minmod4(4.0 * dm1 - d0, 4.0 * d0 - dm1, dm1, d0);                   // Eq. (76), i-1/2
  const double ful = f0 + alpha * dmh;                                                      // Eq. (73)
  const double fmd = 0.5 * (f0 + fp1) - 0.5 * dm4_ph;                                       // Eq. (74)
  const double flc = f0 + 0.5 * dmh + (4.0 / 3.0) * dm4_mh;                                 // Eq. (75)
  const double fmin = std::max(std::min(std::min(f0, fp1), fmd), std::min(std::min(f0, ful), flc));
  const double fmax = std::min(std::max(std::max(f0, fp1), fmd), std::max(std::max(f0, ful), flc));
  return median3(fmin, fhi, fmax);
}

// WENO5 (the second reconstruction the paper names, refs. [61] Shu 1998, [63] Jiang & Shu 1996; the formulas are
// not printed in the paper, this is the textbook scheme of [63] Sec. 3 written out): three third-order candidate values of the
// interface i+1/2, the smoothness indicators IS_k of [63] Eq. (3.1)-(3.3), linear weights (1/10, 6/10, 3/10), exponent 2.
double weno5(double fm2, double fm1, double f0, double fp1, double fp2, double eps) {
  const double q0 = (2.0 * fm2 - 7.0 * fm1 + 11.0 * f0) / 6.0;
  const double q1 = (-fm1 + 5.0 * f0 + 2.0 * fp1) / 6.0;
  const double q2 = (2.0 * f0 + 5.0 * fp1 - fp2) / 6.0;
  const double b0 = 13.0 / 12.0 * (fm2 - 2.0 * fm1 + f0) * (fm2 - 2.0 * fm1 + f0) + 0.25 * (fm2 - 4.0 * fm1 + 3.0 * f0) * (fm2 - 4.0 * fm1 + 3.0 * f0);
  const double b1 = 13.0 / 12.0 * (fm1 - 2.0 * f0 + fp1) * (fm1 - 2.0 * f0 + fp1) + 0.25 * (fm1 - fp1) * (fm1 - fp1);
  const double b2 = 13.0 / 12.0 * (f0 - 2.0 * fp1 + fp2) * (f0 - 2.0 * fp1 + fp2) + 0.25 * (3.0 * f0 - 4.0 * fp1 + fp2) * (3.0 * f0 - 4.0 * fp1 + fp2);
  const double a0 = 0.1 / ((eps + b0) * (eps + b0));
  const double a1 = 0.6 / ((eps + b1) * (eps + b1));
  const double a2 = 0.3 / ((eps + b2) * (eps + b2));
  return (a0 * q0 + a1 * q1 + a2 * q2) / (a0 + a1 + a2);
}

// the reconstruction R of Eq. (66) selected by recon_kind: 0 = MP5 (default, Eqs. 70-76), 1 = WENO5
double reconstruct(const Params& par, double fm2, double fm1, double f0, double fp1, double fp2) {
  if (par.recon_kind == 1) return weno5(fm2, fm1, f0, fp1, fp2, par.weno_eps);
  return mp5(fm2, fm1, f0, fp1, fp2, par.mp5_alpha);
}

}  // namespace orc
