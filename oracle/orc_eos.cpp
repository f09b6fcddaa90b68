// ORACLE (test infrastructure) — equations of state, PAPER.md:236-250 (Eqs. 30-31) and the
// tabulated p(rho,T,Ye), eps(rho,T,Ye) of l.248-250 with reading R26 (trilinear in
// (log10 rho, log10 T, Ye) of log10 p and log10 eps; T from eps by exact inversion of the
// interpolant along the monotone log T axis, clamped to the table).
#include <algorithm>
#include <cmath>
#include "orc.hpp"

namespace orc {

// continuity of eps_cold and p_cold across pieces, PAPER.md:246 (a_0 = 0)
void eos_init(Params& par) {
  if (par.eos_kind != 1) return;
  par.pp_a[0] = 0.0;
  for (int i = 1; i < par.n_pieces; ++i) {
    const double rb = par.pp_rho[i - 1];   // boundary between piece i-1 and i
    // K_i from p continuity: K_{i-1} rb^G_{i-1} = K_i rb^G_i
    par.pp_K[i] = par.pp_K[i - 1] * std::pow(rb, par.pp_Gamma[i - 1] - par.pp_Gamma[i]);
    const double em = par.pp_a[i - 1] + par.pp_K[i - 1] / (par.pp_Gamma[i - 1] - 1.0) * std::pow(rb, par.pp_Gamma[i - 1] - 1.0);
    par.pp_a[i] = em - par.pp_K[i] / (par.pp_Gamma[i] - 1.0) * std::pow(rb, par.pp_Gamma[i] - 1.0);
  }
}

static int pp_piece(const Params& par, double rho) {
  int i = 0;
  while (i < par.n_pieces - 1 && rho >= par.pp_rho[i]) ++i;
  return i;
}
static void pp_cold(const Params& par, double rho, double& pc, double& ec, double& G) {
  const int i = pp_piece(par, rho);
  G = par.pp_Gamma[i];
  const double x = par.pp_K[i] * std::pow(rho, G - 1.0);   // K rho^(G-1) = p_cold / rho
  pc = x * rho;                                            // Eq. (31)
  ec = par.pp_a[i] + x / (G - 1.0);
}

// ---- table helpers ------------------------------------------------------------------
struct TabPos { int i; double w; };
static TabPos tab_locate(double x, double x0, double dx, int n) {
  double s = (x - x0) / dx;
  if (s < 0.0) s = 0.0;
  if (s > (double)(n - 1)) s = (double)(n - 1);
  int i = (int)s;
  if (i > n - 2) i = n - 2;
  return {i, s - (double)i};
}
static size_t tab_idx(const Params& par, int ir, int it, int iy) {
  return ((size_t)iy * par.n_T + it) * par.n_rho + ir;     // rho fastest
}
// bilinear (in log rho, Ye) value of table q at T-node it
static double tab_column(const Params& par, const double* q, TabPos r, TabPos y, int it) {
  const double a = q[tab_idx(par, r.i, it, y.i)], b = q[tab_idx(par, r.i + 1, it, y.i)];
  const double c = q[tab_idx(par, r.i, it, y.i + 1)], d = q[tab_idx(par, r.i + 1, it, y.i + 1)];
  const double lo = a + r.w * (b - a), hi = c + r.w * (d - c);
  return lo + y.w * (hi - lo);
}
static double tab_interp(const Params& par, const double* q, TabPos r, TabPos t, TabPos y) {
  const double lo = tab_column(par, q, r, y, t.i), hi = tab_column(par, q, r, y, t.i + 1);
  return lo + t.w * (hi - lo);
}
// invert log10(eps+shift) -> position on the log T axis (clamped to the table)
static TabPos tab_T_from_loge(const Params& par, TabPos r, TabPos y, double le) {
  int lo = 0, hi = par.n_T - 1;
  const double elo = tab_column(par, par.tab_loge, r, y, lo), ehi = tab_column(par, par.tab_loge, r, y, hi);
  if (le <= elo) return {0, 0.0};
  if (le >= ehi) return {par.n_T - 2, 1.0};
  double e_lo = elo, e_hi = ehi;
  while (hi - lo > 1) {               // bisection on the node index; column is monotone in T
    const int mid = (lo + hi) / 2;
    const double em = tab_column(par, par.tab_loge, r, y, mid);
    if (le >= em) { lo = mid; e_lo = em; } else { hi = mid; e_hi = em; }
  }
  return {lo, (le - e_lo) / (e_hi - e_lo)};
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
