// Bracketing root finder shared by con2prim (App. D) and the M1 closure (Eq. 50).
#pragma once
#include <float.h>
#include <math.h>

namespace mhd {

// Brent's bracketing root finder (the paper's choice, l.1114/l.1143), to ~2 ulp of the root or maxit evaluations.
template <class F>
__device__ double brent_root(F&& fun, double a, double b, double fa, double fb, int maxit, bool& ok) {
  ok = true;
  if (fa == 0.0) return a;
  if (fb == 0.0) return b;
  double c = a, fc = fa, d = b - a, e = d;
  for (int it = 0; it < maxit; ++it) {
    if ((fb > 0.0) == (fc > 0.0)) { c = a; fc = fa; d = b - a; e = d; }
    if (fabs(fc) < fabs(fb)) { a = b; b = c; c = a; fa = fb; fb = fc; fc = fa; }
    const double tol = 2.0 * DBL_EPSILON * fabs(b);
    const double m = 0.5 * (c - b);
    if (fabs(m) <= tol || fb == 0.0) return b;
    if (fabs(e) < tol || fabs(fa) <= fabs(fb)) { d = m; e = m; }
    else {
      double p, q, r, s = fb / fa;
      if (a == c) { p = 2.0 * m * s; q = 1.0 - s; }
      else { q = fa / fc; r = fb / fc; p = s * (2.0 * m * q * (q - r) - (b - a) * (r - 1.0)); q = (q - 1.0) * (r - 1.0) * (s - 1.0); }
      if (p > 0.0) q = -q; else p = -p;
      s = e; e = d;
      if (2.0 * p < 3.0 * m * q - fabs(tol * q) && p < fabs(0.5 * s * q)) d = p / q;
      else { d = m; e = m; }
    }
    a = b; fa = fb;
    b += fabs(d) > tol ? d : (m > 0.0 ? tol : -tol);
    fb = fun(b);
  }
  ok = false;
  return b;
}

}  // namespace mhd
