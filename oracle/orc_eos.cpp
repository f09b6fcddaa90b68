// ORACLE (test infrastructure) — equations of state, PAPER.md:236-250 (Eqs. 30-31) and the
// tabulated p(rho,T,Ye), eps(rho,T,Ye) of l.248-250 with reading R26 (trilinear in
// (log10 rho, log10 T, Ye) of log10 p and log10 eps; T from eps by exact inversion of the
// interpolant along the monotone log T axis, clamped to the table).
// Written the plain way on purpose (8-corner sums, walks over the node coordinates, continuity conditions spelled
// out): the CUDA kernels use nested linear interpolation, index arithmetic and a hinted bisection instead, so a slip in
// either shows up as a parity failure.
#include <algorithm>
#include <cmath>
#include "orc.hpp"

namespace orc {

// Piecewise polytrope, PAPER.md:240-246 (Eq. 31): in piece i (rho_{i-1} <= rho < rho_i)
//     p_cold = K_i rho^Gamma_i,     eps_cold = a_i + K_i rho^(Gamma_i - 1) / (Gamma_i - 1),
// with K_0 given, a_0 = 0, and K_i, a_i (i > 0) fixed by demanding that p_cold and eps_cold are continuous at the
// dividing density rho_{i-1} (l.246). Written out, the two continuity conditions at rb = rho_{i-1} read
//     K_i rb^Gamma_i = p_left,                                where p_left = K_{i-1} rb^Gamma_{i-1},
//     a_i + p_left / ((Gamma_i - 1) rb) = eps_left,            where eps_left = a_{i-1} + p_left / ((Gamma_{i-1} - 1) rb),
// (using K rho^(Gamma-1) = p_cold / rho on both sides of the second one).
void eos_init(Params& par) {
  if (par.eos_kind != 1) return;
  par.pp_a[0] = 0.0;
  for (int i = 1; i < par.n_pieces; ++i) {
    const double rb = par.pp_rho[i - 1];
    const double p_left = par.pp_K[i - 1] * std::exp(par.pp_Gamma[i - 1] * std::log(rb));
    const double eps_left = par.pp_a[i - 1] + p_left / ((par.pp_Gamma[i - 1] - 1.0) * rb);
    par.pp_K[i] = p_left / std::exp(par.pp_Gamma[i] * std::log(rb));
    par.pp_a[i] = eps_left - p_left / ((par.pp_Gamma[i] - 1.0) * rb);
  }
}

// cold pressure, cold specific internal energy and exponent of the piece that contains rho
static void pp_cold(const Params& par, double rho, double& pc, double& ec, double& G) {
  int piece = par.n_pieces - 1;                              // the last piece is unbounded above
  for (int i = par.n_pieces - 2; i >= 0; --i)                // walk down while rho lies below the dividing density
    if (rho < par.pp_rho[i]) piece = i;
  G = par.pp_Gamma[piece];
  pc = par.pp_K[piece] * std::pow(rho, G);                   // Eq. (31)
  ec = par.pp_a[piece] + pc / ((G - 1.0) * rho);
}

// ---- table (R26): values on the nodes x_i = x0 + i dx of the three axes (log10 rho, log10 T, Ye), rho fastest -------------
static double tab_node(const Params& par, const double* q, int ir, int it, int iy) {
  return q[((size_t)iy * par.n_T + it) * par.n_rho + ir];
}
// cell [x_i, x_{i+1}] holding x and the weight of its upper node; x is clamped to the table first. Found by walking along
// the node coordinates themselves.
struct TabPos { int i; double w; };
static TabPos tab_locate(double x, double x0, double dx, int n) {
  const double xlast = x0 + (n - 1) * dx;
  if (x <= x0) return {0, 0.0};
  if (x >= xlast) return {n - 2, 1.0};
  int i = 0;
  while (i < n - 2 && x >= x0 + (i + 1) * dx) ++i;
  double w = (x - (x0 + i * dx)) / dx;
  if (w < 0.0) w = 0.0;
  if (w > 1.0) w = 1.0;
  return {i, w};
}
// PAPER.md:250 "linear interpolation": the trilinear interpolant is the sum over the 8 corners of the cell, each weighted by
// the product of its three one-dimensional weights
static double tab_interp(const Params& par, const double* q, TabPos r, TabPos t, TabPos y) {
  double sum = 0.0;
  for (int cy = 0; cy < 2; ++cy)
    for (int ct = 0; ct < 2; ++ct)
      for (int cr = 0; cr < 2; ++cr) {
        const double w = (cr ? r.w : 1.0 - r.w) * (ct ? t.w : 1.0 - t.w) * (cy ? y.w : 1.0 - y.w);
        sum += w * tab_node(par, q, r.i + cr, t.i + ct, y.i + cy);
      }
  return sum;
}
// the interpolant on the T node `it` (weight 1 on that node): the 4-corner sum in (log10 rho, Ye)
static double tab_column(const Params& par, const double* q, TabPos r, TabPos y, int it) {
  const TabPos on_node = {it < par.n_T - 1 ? it : it - 1, it < par.n_T - 1 ? 0.0 : 1.0};
  return tab_interp(par, q, r, on_node, y);
}
// T from eps at fixed (rho, Ye): the interpolant is piecewise linear and increasing along the log10 T axis, so its inverse
// is found by walking up the T nodes until the column value exceeds log10(eps + shift) (coarse strides of 16 nodes first,
// then node by node), and solving the linear interpolation in that cell. Below / above the table: clamped (l.1145).
static TabPos tab_T_from_loge(const Params& par, TabPos r, TabPos y, double le) {
  const int last = par.n_T - 1;
  if (le <= tab_column(par, par.tab_loge, r, y, 0)) return {0, 0.0};
  if (le >= tab_column(par, par.tab_loge, r, y, last)) return {last - 1, 1.0};
  int it = 0;
  while (it + 16 < last && le >= tab_column(par, par.tab_loge, r, y, it + 16)) it += 16;
  while (it + 1 < last && le >= tab_column(par, par.tab_loge, r, y, it + 1)) ++it;
  const double e_lo = tab_column(par, par.tab_loge, r, y, it), e_hi = tab_column(par, par.tab_loge, r, y, it + 1);
  return {it, (le - e_lo) / (e_hi - e_lo)};
}

// slope of the trilinear interpolant of table q along one axis (0: log10 rho, 1: log10 T, 2: Ye) inside the cell (r, t, y): the difference of the
// two faces of the cell across that axis, each face bilinear in the other two variables, over the node spacing
static double tab_slope(const Params& par, const double* q, TabPos r, TabPos t, TabPos y, int axis) {
  double sum = 0.0;
  for (int c1 = 0; c1 < 2; ++c1)
    for (int c2 = 0; c2 < 2; ++c2) {
      double w, hi, lo;
      if (axis == 0) { w = (c1 ? t.w : 1.0 - t.w) * (c2 ? y.w : 1.0 - y.w); hi = tab_node(par, q, r.i + 1, t.i + c1, y.i + c2); lo = tab_node(par, q, r.i, t.i + c1, y.i + c2); }
      else if (axis == 1) { w = (c1 ? r.w : 1.0 - r.w) * (c2 ? y.w : 1.0 - y.w); hi = tab_node(par, q, r.i + c1, t.i + 1, y.i + c2); lo = tab_node(par, q, r.i + c1, t.i, y.i + c2); }
      else { w = (c1 ? r.w : 1.0 - r.w) * (c2 ? t.w : 1.0 - t.w); hi = tab_node(par, q, r.i + c1, t.i + c2, y.i + 1); lo = tab_node(par, q, r.i + c1, t.i + c2, y.i); }
      sum += w * (hi - lo);
    }
  return sum / (axis == 0 ? par.dlr : axis == 1 ? par.dlT : par.dye);
}

// dp/drho at fixed (eps, Ye), dp/deps at fixed (rho, Ye), dp/dYe at fixed (rho, eps) (App. A, l.882: "analytically for hybrid EoSs, but only
// numerically for the tabulated ones"). Table (reading R42): the derivatives of the interpolant itself inside the cell that holds (rho, T, Ye) —
// with lp = log10 p, le = log10(eps + shift) trilinear in (lr, lT, Ye):  d lp/d lr at fixed le = lp_r - lp_T le_r / le_T,  d lp/d le at fixed lr =
// lp_T / le_T,  d lp/d Ye at fixed (lr, le) = lp_Y - lp_T le_Y / le_T;  then dp/drho = (p/rho) d lp/d lr, dp/deps = p/(eps + shift) d lp/d le,
// dp/dYe = p ln 10 d lp/d Ye.
void eos_dp(const Params& par, double rho, double eps, double ye, double& dpdrho, double& dpdeps, double& dpdye) {
  dpdye = 0.0;
  if (par.eos_kind == 0) { dpdrho = (par.eos_gamma - 1.0) * eps; dpdeps = (par.eos_gamma - 1.0) * rho; return; }
  if (par.eos_kind == 1) {
    // p = p_cold + (Gamma_th - 1) rho (eps - eps_cold) (Eq. 30), d p_cold / d rho = Gamma_i p_cold / rho, d eps_cold / d rho = p_cold / rho^2
    double pc, ec, G;
    pp_cold(par, rho, pc, ec, G);
    const double gth = par.eos_gamma_th - 1.0;
    dpdrho = G * pc / rho + gth * (eps - ec) - gth * pc / rho;
    dpdeps = gth * rho;
    return;
  }
  const TabPos r = tab_locate(std::log10(rho), par.lr0, par.dlr, par.n_rho);
  const TabPos y = tab_locate(ye, par.ye0, par.dye, par.n_ye);
  const TabPos t = tab_T_from_loge(par, r, y, std::log10(eps + par.tab_eps_shift));
  const double p = std::pow(10.0, tab_interp(par, par.tab_logp, r, t, y));
  const double lp_r = tab_slope(par, par.tab_logp, r, t, y, 0), lp_T = tab_slope(par, par.tab_logp, r, t, y, 1), lp_Y = tab_slope(par, par.tab_logp, r, t, y, 2);
  const double le_r = tab_slope(par, par.tab_loge, r, t, y, 0), le_T = tab_slope(par, par.tab_loge, r, t, y, 1), le_Y = tab_slope(par, par.tab_loge, r, t, y, 2);
  dpdrho = p / rho * (lp_r - lp_T * le_r / le_T);
  dpdeps = p / (eps + par.tab_eps_shift) * (lp_T / le_T);
  dpdye = p * std::log(10.0) * (lp_Y - lp_T * le_Y / le_T);
}

EosOut eos_from_rho_eps(const Params& par, double rho, double eps, double ye) {
  EosOut o;
  if (par.eos_kind == 0) {
    o.p = (par.eos_gamma - 1.0) * rho * eps;               // ideal gas
    o.T = o.p / rho;                                        // R27: synthetic temperature p/rho
    const double h = 1.0 + eps + o.p / rho;                 // specific enthalpy
    o.cs2 = par.eos_gamma * o.p / (rho * h);                // PAPER.md:905  cs^2 = Gamma p / h
    return o;
  }
  if (par.eos_kind == 1) {
    double pc, ec, G;
    pp_cold(par, rho, pc, ec, G);
    const double gth = par.eos_gamma_th - 1.0;
    o.p = pc + gth * rho * (eps - ec);                      // Eq. (30) with p_th = (Gamma_th-1) rho eps_th
    o.T = o.p / rho;
    const double h = 1.0 + eps + o.p / rho;
    // R13: cs^2 = (dp/drho|eps + p/rho^2 dp/deps|rho) / h,  d eps_cold/d rho = p_cold / rho^2
    const double dpdrho = G * pc / rho + gth * (eps - ec) - gth * pc / rho;
    const double dpdeps = gth * rho;
    o.cs2 = (dpdrho + o.p / (rho * rho) * dpdeps) / h;
    return o;
  }
  const TabPos r = tab_locate(std::log10(rho), par.lr0, par.dlr, par.n_rho);
  const TabPos y = tab_locate(ye, par.ye0, par.dye, par.n_ye);
  const TabPos t = tab_T_from_loge(par, r, y, std::log10(eps + par.tab_eps_shift));
  o.p = std::pow(10.0, tab_interp(par, par.tab_logp, r, t, y));
  o.T = std::pow(10.0, par.lT0 + ((double)t.i + t.w) * par.dlT);
  o.cs2 = tab_interp(par, par.tab_cs2, r, t, y);
  return o;
}

double eos_eps_from_T(const Params& par, double rho, double T, double ye) {
  const TabPos r = tab_locate(std::log10(rho), par.lr0, par.dlr, par.n_rho);
  const TabPos y = tab_locate(ye, par.ye0, par.dye, par.n_ye);
  const TabPos t = tab_locate(std::log10(T), par.lT0, par.dlT, par.n_T);
  return std::pow(10.0, tab_interp(par, par.tab_loge, r, t, y)) - par.tab_eps_shift;
}

// validity region
void eos_eps_range(const Params& par, double rho, double ye, double& emin, double& emax) {
  if (par.eos_kind == 0) { emin = par.eps_min; emax = par.eps_max; return; }
  if (par.eos_kind == 1) {
    double pc, ec, G;
    pp_cold(par, rho, pc, ec, G);
    emin = std::max(par.eps_min, ec);   // eps_th >= 0
    emax = par.eps_max;
    return;
  }
  const TabPos r = tab_locate(std::log10(rho), par.lr0, par.dlr, par.n_rho);
  const TabPos y = tab_locate(ye, par.ye0, par.dye, par.n_ye);
  emin = std::pow(10.0, tab_column(par, par.tab_loge, r, y, 0)) - par.tab_eps_shift;
  emax = std::pow(10.0, tab_column(par, par.tab_loge, r, y, par.n_T - 1)) - par.tab_eps_shift;
}

void eos_rho_range(const Params& par, double& rmin, double& rmax) {
  if (par.eos_kind == 2) {
    rmin = std::pow(10.0, par.lr0);
    rmax = std::pow(10.0, par.lr0 + par.dlr * (par.n_rho - 1));
  } else { rmin = 0.0; rmax = par.rho_max; }
}

// R8: lower bound of the specific relativistic enthalpy over the validity region
double eos_h0(const Params& par) { return par.eos_kind == 2 ? par.tab_h0 : 1.0; }

}  // namespace orc
