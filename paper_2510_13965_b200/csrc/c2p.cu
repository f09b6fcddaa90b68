// a2 — conserved -> primitive recovery at every grid point (App. D, Eqs. D1-D15; error policy
// l.1157-1162) and its inverse for initial data (Eq. 29), with the three equations of state
// (ideal gas, hybrid piecewise polytrope Eqs. 30-31, tabulated p/eps(rho,T,Ye) l.248-250).
//
// Flag reproducibility (DESIGN.md note N2): the atmosphere decision is taken on D = Dbar * (chi * sqrt(chi)) —
// multiplications and one square root only, so no FMA can form and the result is the IEEE value the oracle
// computes. Every other rule of the error policy acts on the output of the root solve, which is defined only up to
// its tolerance; inputs keep away from those thresholds. Divisions are hoisted into reciprocals (one per
// denominator) because an FP64 division costs about ten FP64-pipe instructions.
//
// Warp-divergence control: a CTA owns a chunk of C2P_CHUNK consecutive points. Pass A decides "atmosphere" for every point
// of the chunk (the contraction-free pre-check), writes the atmosphere state of those points at once (the same for every
// such cell: its EoS part is computed once per launch by k_atmo_state) and compacts the indices of the others into a
// shared-memory list (ballot + one atomic per warp). Pass B runs the App. D solve on that list, 32 live lanes per warp,
// so the cells at the stellar surface do not share warps with atmosphere cells that have nothing to do. Both root solves
// are bounded by c2p_maxit.
// Tabulated EoS inside the mu iteration: Ye is fixed during the solve, so each thread keeps the Ye-collapsed corner values
// of the (log10 rho, log10 T) cell it is in (4 of log10 eps, 4 of log10 p). As long as the iterate stays in that cell an
// evaluation of p(rho, eps) is two log10, one exp10 and a dozen FMAs with no memory access; a change of cell re-runs the
// search (the interpolant is monotone along T, so whatever the search order the cell found is the same).
#include <float.h>
#include "mhd_internal.cuh"
#include "rootfind.cuh"

namespace mhd {

// ------------------------------------------------------------------------------------------ EoS
struct Eos { double p, T, cs2; };

// The library's log10 / exp10 expand to ~100 instructions each. con2prim is bound by instruction fetch (long straight-line code
// run once per cell), so every call site shares ONE out-of-line copy.
__device__ __noinline__ double log10_1(double x) { return log10(x); }
__device__ __noinline__ double exp10_1(double x) { return exp10(x); }

__device__ __forceinline__ int pp_piece(const Par& q, double rho) {
  int i = 0;
  while (i < q.n_pieces - 1 && rho >= q.pp_rho[i]) ++i;
  return i;
}
__device__ __forceinline__ void pp_cold(const Par& q, double rho, double& pc, double& ec, double& G) {
  const int i = pp_piece(q, rho);
  G = q.pp_Gamma[i];
  const double x = q.pp_K[i] * pow(rho, G - 1.0);
  pc = x * rho;
  ec = q.pp_a[i] + x / (G - 1.0);
}

struct TPos { int i; double w; };
__device__ __forceinline__ TPos tab_locate(double x, double x0, double idx, int n) {      // idx = 1 / spacing
  double s = (x - x0) * idx;
  s = fmin(fmax(s, 0.0), (double)(n - 1));
  int i = (int)s;
  if (i > n - 2) i = n - 2;
  TPos r; r.i = i; r.w = s - (double)i;
  return r;
}
// bilinear (log rho, Ye) value of table t at T node it; the 4 gathers hit L2 (tables are <= 10 MB each)
__device__ __forceinline__ double tab_col(const Par& q, const double* __restrict__ t, TPos r, TPos y, int it) {
  const size_t b0 = ((size_t)y.i * q.n_T + it) * q.n_rho + r.i;
  const size_t b1 = b0 + (size_t)q.n_T * q.n_rho;
  const double a = __ldg(t + b0), b = __ldg(t + b0 + 1), c = __ldg(t + b1), d = __ldg(t + b1 + 1);
  const double lo = a + r.w * (b - a), hi = c + r.w * (d - c);
  return lo + y.w * (hi - lo);
}
__device__ __forceinline__ double tab_tri(const Par& q, const double* __restrict__ t, TPos r, TPos tt, TPos y) {
  const double lo = tab_col(q, t, r, y, tt.i), hi = tab_col(q, t, r, y, tt.i + 1);
  return lo + tt.w * (hi - lo);
}
// exact inverse of the interpolant along the (monotone) log T axis, clamped to the table
__device__ __forceinline__ TPos tab_T_of_loge(const Par& q, TPos r, TPos y, double le) {
  int lo = 0, hi = q.n_T - 1;
  double e_lo = tab_col(q, q.tab_loge, r, y, lo), e_hi = tab_col(q, q.tab_loge, r, y, hi);
  TPos o;
  if (le <= e_lo) { o.i = 0; o.w = 0.0; return o; }
  if (le >= e_hi) { o.i = q.n_T - 2; o.w = 1.0; return o; }
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    const double em = tab_col(q, q.tab_loge, r, y, mid);
    if (le >= em) { lo = mid; e_lo = em; } else { hi = mid; e_hi = em; }
  }
  o.i = lo; o.w = (le - e_lo) / (e_hi - e_lo);
  return o;
}

template <int KIND>
__device__ __forceinline__ Eos eos_eval(const Par& q, double rho, double eps, double ye) {
  Eos o;
  if (KIND == 0) {
    o.p = (q.eos_gamma - 1.0) * rho * eps;
    o.T = o.p / rho;
    const double h = 1.0 + eps + o.p / rho;
    o.cs2 = q.eos_gamma * o.p / (rho * h);
  } else if (KIND == 1) {
    double pc, ec, G;
    pp_cold(q, rho, pc, ec, G);
    const double gth = q.eos_gamma_th - 1.0;
    o.p = pc + gth * rho * (eps - ec);
    o.T = o.p / rho;
    const double h = 1.0 + eps + o.p / rho;
    const double dpdrho = G * pc / rho + gth * (eps - ec) - gth * pc / rho;
    o.cs2 = (dpdrho + o.p / (rho * rho) * (gth * rho)) / h;
  } else {
    const TPos r = tab_locate(log10_1(rho), q.lr0, q.idlr, q.n_rho);
    const TPos y = tab_locate(ye, q.ye0, q.idye, q.n_ye);
    const TPos t = tab_T_of_loge(q, r, y, log10_1(eps + q.tab_eps_shift));
    o.p = exp10_1(tab_tri(q, q.tab_logp, r, t, y));
    o.T = exp10_1(q.lT0 + ((double)t.i + t.w) * q.dlT);
    o.cs2 = tab_tri(q, q.tab_cs2, r, t, y);
  }
  return o;
}
template <int KIND>
__device__ __forceinline__ void eos_eps_range(const Par& q, double rho, double ye, double& emin, double& emax) {
  if (KIND == 0) { emin = q.eps_min; emax = q.eps_max; }
  else if (KIND == 1) {
    double pc, ec, G;
    pp_cold(q, rho, pc, ec, G);
    emin = fmax(q.eps_min, ec); emax = q.eps_max;
  } else {
    const TPos r = tab_locate(log10_1(rho), q.lr0, q.idlr, q.n_rho);
    const TPos y = tab_locate(ye, q.ye0, q.idye, q.n_ye);
    emin = exp10_1(tab_col(q, q.tab_loge, r, y, 0)) - q.tab_eps_shift;
    emax = exp10_1(tab_col(q, q.tab_loge, r, y, q.n_T - 1)) - q.tab_eps_shift;
  }
}
__device__ __forceinline__ double eos_eps_of_T(const Par& q, double rho, double T, double ye) {
  const TPos r = tab_locate(log10_1(rho), q.lr0, q.idlr, q.n_rho);
  const TPos y = tab_locate(ye, q.ye0, q.idye, q.n_ye);
  const TPos t = tab_locate(log10_1(T), q.lT0, q.idlT, q.n_T);
  return exp10_1(tab_tri(q, q.tab_loge, r, t, y)) - q.tab_eps_shift;
}

// ------------------------------------------------------------------------------------------ metric helpers
struct Sym3 { double xx, xy, xz, yy, yz, zz; };
__device__ __forceinline__ void sym_apply(const Sym3& g, const double v[3], double o[3]) {
  o[0] = g.xx * v[0] + g.xy * v[1] + g.xz * v[2];
  o[1] = g.xy * v[0] + g.yy * v[1] + g.yz * v[2];
  o[2] = g.xz * v[0] + g.yz * v[1] + g.zz * v[2];
}
// inverse times the factor s
__device__ __forceinline__ Sym3 sym_inverse(const Sym3& g, double s) {
  const double det = g.xx * (g.yy * g.zz - g.yz * g.yz) - g.xy * (g.xy * g.zz - g.yz * g.xz) + g.xz * (g.xy * g.yz - g.yy * g.xz);
  const double f = s / det;
  Sym3 r;
  r.xx = (g.yy * g.zz - g.yz * g.yz) * f;
  r.xy = (g.xz * g.yz - g.xy * g.zz) * f;
  r.xz = (g.xy * g.yz - g.xz * g.yy) * f;
  r.yy = (g.xx * g.zz - g.xz * g.xz) * f;
  r.yz = (g.xy * g.xz - g.xx * g.yz) * f;
  r.zz = (g.xx * g.yy - g.xy * g.xy) * f;
  return r;
}
__device__ __forceinline__ Sym3 sym_scale(const Sym3& g, double s) {
  Sym3 r;
  r.xx = s * g.xx; r.xy = s * g.xy; r.xz = s * g.xz; r.yy = s * g.yy; r.yz = s * g.yz; r.zz = s * g.zz;
  return r;
}

// Eq. (29): undensitised D, tau, S_i from primitives (h = enthalpy density)
__device__ __forceinline__ void cons_from_prim(const Sym3& gl, double rho, double eps, double p, const double v[3],
                                               const double B[3], double& D, double& tau, double S[3], double& W) {
  double vl[3], Bl[3];
  sym_apply(gl, v, vl);
  sym_apply(gl, B, Bl);
  const double v2 = v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2];
  const double B2 = B[0] * Bl[0] + B[1] * Bl[1] + B[2] * Bl[2];
  const double Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2];
  const double W2 = 1.0 / (1.0 - v2);
  W = sqrt(W2);
  const double h = rho * (1.0 + eps) + p;
  D = rho * W;
  tau = h * W2 - p + B2 - 0.5 * (Bv * Bv + B2 / W2) - D;
#pragma unroll
  for (int i = 0; i < 3; ++i) S[i] = (h * W2 + B2) * vl[i] - Bv * Bl[i];
}

// ------------------------------------------------------------------------------------------ root solves
// Per-thread cache of the table cell of the last evaluation (see the header): Ye-collapsed corner values, [T node][rho node].
struct TabCell {
  int ir, it;            // cell indices; ir = -1: empty
  double e[2][2], p[2][2];
};
__device__ __forceinline__ double ye_collapse(const Par& q, const double* __restrict__ t, TPos y, int it, int ir) {
  const size_t b0 = ((size_t)y.i * q.n_T + it) * q.n_rho + ir;
  const double a = __ldg(t + b0), c = __ldg(t + b0 + (size_t)q.n_T * q.n_rho);
  return a + y.w * (c - a);
}
__device__ __forceinline__ void tab_cell_fill(const Par& q, TPos y, int ir, int it, TabCell& c) {
  c.ir = ir; c.it = it;
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      c.e[a][b] = ye_collapse(q, q.tab_loge, y, it + a, ir + b);
      c.p[a][b] = ye_collapse(q, q.tab_logp, y, it + a, ir + b);
    }
}
// column value (T node it) of log10 eps at the Ye-collapsed rho position r
__device__ __forceinline__ double tab_ecol(const Par& q, TPos r, TPos y, int it) {
  const double a = ye_collapse(q, q.tab_loge, y, it, r.i), b = ye_collapse(q, q.tab_loge, y, it, r.i + 1);
  return a + r.w * (b - a);
}
// cell search along T for log10_1(eps + shift) = le, with the clamps of l.1145; returns the T position, sets clamp = -1 / +1 / 0
struct TSearch { double w; int i, clamp; };
__device__ __noinline__ TSearch tab_T_search(const Par& q, TPos r, TPos y, double le, int hint) {
  TSearch t;
  const double e_min = tab_ecol(q, r, y, 0), e_max = tab_ecol(q, r, y, q.n_T - 1);
  if (!(le > e_min)) { t.i = 0; t.w = 0.0; t.clamp = -1; return t; }
  if (le >= e_max) { t.i = q.n_T - 2; t.w = 1.0; t.clamp = 1; return t; }
  t.clamp = 0;
  int lo = 0, hi = q.n_T - 1;
  double e_lo = e_min, e_hi = e_max;
  if (hint >= 0 && hint < q.n_T - 1) {               // the hinted cell, then its neighbours, then bisection
    const double a = tab_ecol(q, r, y, hint), b = tab_ecol(q, r, y, hint + 1);
    if (le >= a) { lo = hint; e_lo = a; if (le < b) { hi = hint + 1; e_hi = b; } else { lo = hint + 1; e_lo = b; } }
    else { hi = hint; e_hi = a; }
  }
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    const double em = tab_ecol(q, r, y, mid);
    if (le >= em) { lo = mid; e_lo = em; } else { hi = mid; e_hi = em; }
  }
  t.i = lo; t.w = (le - e_lo) / (e_hi - e_lo);
  return t;
}
// log10 and 10^x of an argument that stays close to a reference (the iterates of one root solve move by << 1e-3): the Taylor
// series about the reference, five terms, truncation error below 2^-60 relative for |t| < 2^-10 — the same double-precision value
// as the library routine (which costs ~10x more FP64 instructions); outside that range the library routine sets a new reference.
struct LogRef { double x, ix, l; };        // reference argument, its reciprocal, log10_1(reference); x = 0: empty
__device__ __forceinline__ double log10_near(double x, LogRef& r) {
  const double t = (x - r.x) * r.ix;
  if (fabs(t) < 0x1p-10) {
    const double c1 = 0.43429448190325182765, c2 = -0.5 * c1, c3 = c1 / 3.0, c4 = -0.25 * c1, c5 = 0.2 * c1;   // (-1)^(k+1) / (k ln 10)
    return fma(t, fma(t, fma(t, fma(t, fma(t, c5, c4), c3), c2), c1), r.l);
  }
  r.x = x; r.ix = 1.0 / x; r.l = log10_1(x);
  return r.l;
}
struct ExpRef { double l, p; };            // reference exponent and 10^l
__device__ __forceinline__ double exp10_near(double l, ExpRef& r) {
  const double y = (l - r.l) * 2.30258509299404568402;
  if (fabs(y) < 0x1p-9) return r.p * fma(y, fma(y, fma(y, fma(y, fma(y, 1.0 / 120.0, 1.0 / 24.0), 1.0 / 6.0), 0.5), 1.0), 1.0);
  r.l = l; r.p = exp10_1(l);
  return r.p;
}
struct TabState {                          // everything the table path carries from one evaluation of f to the next
  TabCell cell;
  LogRef lrho, leps;
  ExpRef lp;
  int hint;
  int clamp;                               // -1 / +1: the last evaluation clamped eps to the lower / upper edge of the table (l.1145)
  TPos tpos, rpos;                         // table position of the last evaluation
};

// Tabulated EoS inside the mu iteration: pressure and clamped eps for (rho, eps_raw) at fixed Ye.
__device__ __forceinline__ void tab_p_of_eps(const Par& q, TPos y, double rho, double eps_raw, TabState& ts, double& p, double& eps) {
  TabCell& c = ts.cell;
  const TPos r = tab_locate(log10_near(rho, ts.lrho), q.lr0, q.idlr, q.n_rho);
  const double ea = eps_raw + q.tab_eps_shift;
  const double le = ea > 0.0 ? log10_near(ea, ts.leps) : -INFINITY;
  ts.rpos = r;
  eps = eps_raw;
  if (r.i == c.ir) {                                  // fast path: still in the cached cell?
    const double e_lo = c.e[0][0] + r.w * (c.e[0][1] - c.e[0][0]), e_hi = c.e[1][0] + r.w * (c.e[1][1] - c.e[1][0]);
    if (le >= e_lo && le < e_hi) {
      ts.tpos.i = c.it; ts.tpos.w = (le - e_lo) / (e_hi - e_lo);
      const double p_lo = c.p[0][0] + r.w * (c.p[0][1] - c.p[0][0]), p_hi = c.p[1][0] + r.w * (c.p[1][1] - c.p[1][0]);
      p = exp10_near(p_lo + ts.tpos.w * (p_hi - p_lo), ts.lp);
      ts.clamp = 0;
      return;
    }
  }
  const TSearch found = tab_T_search(q, r, y, le, ts.hint);
  const int clamp = found.clamp;
  ts.clamp = clamp;
  ts.tpos.i = found.i; ts.tpos.w = found.w;
  ts.hint = ts.tpos.i;
  tab_cell_fill(q, y, r.i, ts.tpos.i, c);
  const double e_lo = c.e[0][0] + r.w * (c.e[0][1] - c.e[0][0]), e_hi = c.e[1][0] + r.w * (c.e[1][1] - c.e[1][0]);
  if (clamp < 0) eps = exp10_1(e_lo) - q.tab_eps_shift;
  else if (clamp > 0) eps = exp10_1(e_hi) - q.tab_eps_shift;
  const double p_lo = c.p[0][0] + r.w * (c.p[0][1] - c.p[0][0]), p_hi = c.p[1][0] + r.w * (c.p[1][1] - c.p[1][0]);
  p = exp10_near(p_lo + ts.tpos.w * (p_hi - p_lo), ts.lp);
}

template <int KIND>
struct Master {
  double D, q, r2, B2, rB2, B2rp2, ye, h0, v02, rho_lo, rho_hi;
  double W, eps_raw;   // by-products of the last evaluation
  double p_last;       // pressure of the last evaluation
  TPos ypos;           // table position of Ye (fixed during the solve)
  TabState tab;        // KIND 2
  __device__ __forceinline__ double x_of(double mu) const { return 1.0 / (1.0 + mu * B2); }          // (D5)
  __device__ __forceinline__ double rbar2(double mu) const {                                          // (D4)
    const double x = x_of(mu);
    return r2 * x * x + mu * x * (1.0 + x) * rB2;
  }
  __device__ __forceinline__ double fa(double mu) const { return mu * sqrt(h0 * h0 + rbar2(mu)) - 1.0; }   // (D3)
  __device__ __forceinline__ double f(const Par& par, double mu) {                                        // (D6)-(D14)
    const double x = x_of(mu);
    const double rb2 = r2 * x * x + mu * x * (1.0 + x) * rB2;
    const double qbar = q - 0.5 * B2 - 0.5 * mu * mu * x * x * B2rp2;
    const double v2 = fmin(mu * mu * rb2, v02);
    const double iW = sqrt(1.0 - v2);
    W = 1.0 / iW;
    double rho = D * iW;
    rho = fmax(fmin(rho_hi, rho), rho_lo);
    eps_raw = W * ((qbar - mu * rb2) + v2 / (1.0 + iW));                                             // (D12): W^2/(1+W) = W/(1+1/W)
    double eps, p;
    if (KIND == 2) tab_p_of_eps(par, ypos, rho, eps_raw, tab, p, eps);
    else {
      double emin, emax;
      eos_eps_range<KIND>(par, rho, ye, emin, emax);
      eps = fmax(fmin(emax, eps_raw), emin);
      p = eos_eval<KIND>(par, rho, eps, ye).p;
    }
    p_last = p;
    const double a = p / (rho * (1.0 + eps));
    const double nuA = (1.0 + a) * (1.0 + eps) * iW;
    const double nuB = (1.0 + a) * (1.0 + qbar - mu * rb2);
    return mu - 1.0 / (fmax(nuA, nuB) + mu * rb2);
  }
};

// ------------------------------------------------------------------------------------------ kernels
constexpr int C2P_THREADS = 128, C2P_PER_THREAD = 4, C2P_CHUNK = C2P_THREADS * C2P_PER_THREAD;

// EoS part of the atmosphere state (rule 1 of l.1157): eps, p, T, cs2 at (rho_atmo, T_atmo | eps_atmo, Ye_atmo). The same for every
// atmosphere cell, so it is evaluated once per launch by one thread instead of once per cell.
template <int KIND>
__global__ void k_atmo_state(const __grid_constant__ Par par, double* __restrict__ out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const double rho = par.rho_atmo, ye = par.ye_atmo;
  double eps;
  if (KIND == 2) eps = eos_eps_of_T(par, rho, par.T_atmo, ye);
  else if (KIND == 1) { double emin, emax; eos_eps_range<KIND>(par, rho, ye, emin, emax); eps = emin + par.eps_atmo; }
  else eps = par.eps_atmo;
  const Eos e = eos_eval<KIND>(par, rho, eps, ye);
  out[0] = eps; out[1] = e.p; out[2] = e.T; out[3] = e.cs2;
}

struct C2pIo {
  double* U; size_t su; double* P; size_t sp; uint8_t* flags;
};

__device__ __forceinline__ void store_point(const C2pIo& io, long long pt, const Sym3& gl, double sg, const double B[3], double rho, double ye,
                                            double eps, const Eos& e, const double v[3], double W, unsigned flag, bool changed) {
  double* P = io.P;
  const size_t sp = io.sp;
  P[(size_t)RHO * sp + pt] = rho; P[(size_t)YE * sp + pt] = ye; P[(size_t)EPS * sp + pt] = eps; P[(size_t)PRESS * sp + pt] = e.p;
  P[(size_t)VX * sp + pt] = v[0]; P[(size_t)VY * sp + pt] = v[1]; P[(size_t)VZ * sp + pt] = v[2];
  P[(size_t)WLOR * sp + pt] = W; P[(size_t)TEMP * sp + pt] = e.T; P[(size_t)CS2 * sp + pt] = e.cs2;
  io.flags[pt] = (uint8_t)flag;
  if (changed) {                                                                     // R11
    double Dn, taun, Sn[3], Wn;
    cons_from_prim(gl, rho, eps, e.p, v, B, Dn, taun, Sn, Wn);
    double* U = io.U;
    const size_t su = io.su;
    U[(size_t)DBAR * su + pt] = sg * Dn; U[(size_t)DYEBAR * su + pt] = sg * Dn * ye; U[(size_t)TAUBAR * su + pt] = sg * taun;
    U[(size_t)SXBAR * su + pt] = sg * Sn[0]; U[(size_t)SYBAR * su + pt] = sg * Sn[1]; U[(size_t)SZBAR * su + pt] = sg * Sn[2];
  }
}

// rule 1: reset to atmosphere
__device__ __forceinline__ void store_atmosphere(const C2pIo& io, const Par& par, long long pt, const double* __restrict__ atmo, unsigned flag) {
  auto u = [&](int f) { return io.U[(size_t)f * io.su + pt]; };
  const Sym3 gt = {u(GXX), u(GXY), u(GXZ), u(GYY), u(GYZ), u(GZZ)};
  const double chi = u(CHI);
  const double isg = chi * sqrt(chi), sg = 1.0 / isg;
  const Sym3 gl = sym_scale(gt, 1.0 / chi);
  const double B[3] = {u(BXBAR) * isg, u(BYBAR) * isg, u(BZBAR) * isg};
  const double v[3] = {0.0, 0.0, 0.0};
  Eos e;
  e.p = __ldg(atmo + 1); e.T = __ldg(atmo + 2); e.cs2 = __ldg(atmo + 3);
  store_point(io, pt, gl, sg, B, par.rho_atmo, par.ye_atmo, __ldg(atmo), e, v, 1.0, flag | MHD_FLAG_ATMO, true);
}

// App. D steps 1-4 and the error policy for one point that passed the atmosphere pre-check
template <int KIND>
__device__ __forceinline__ void solve_point(const C2pIo& io, const Par& par, long long pt, const double* __restrict__ atmo) {
  auto u = [&](int f) { return io.U[(size_t)f * io.su + pt]; };
  const double* P = io.P;
  const size_t sp = io.sp;
  const Sym3 gt = {u(GXX), u(GXY), u(GXZ), u(GYY), u(GYZ), u(GZZ)};
  const double chi = u(CHI), alpha = u(ALPHA);
  const double Dbar = u(DBAR), DYe = u(DYEBAR);
  const double isg = chi * sqrt(chi);            // 1/sqrt(gamma) = chi^(3/2)   (det gamma~ = 1)
  const double sg = 1.0 / isg;
  const double D = Dbar * isg;                   // note N2: mul, sqrt, mul only
  const Sym3 gl = sym_scale(gt, 1.0 / chi);      // gamma_ij = gamma~_ij / chi
  const Sym3 gu = sym_inverse(gt, chi);          // gamma^ij = chi gamma~^ij
  const double B[3] = {u(BXBAR) * isg, u(BYBAR) * isg, u(BZBAR) * isg};
  double ye = DYe / Dbar;
  unsigned int flag = 0;
  double rho, eps, W, v[3];
  bool changed = false;
  const bool bh = alpha < par.alpha_bh;

  const double tau = u(TAUBAR) * isg;
  const double Sl[3] = {u(SXBAR) * isg, u(SYBAR) * isg, u(SZBAR) * isg};
  Master<KIND> s;
  const double iD = 1.0 / D, isD = 1.0 / sqrt(D);
  s.D = D; s.q = tau * iD;                                                         // (D1)
  const double rl[3] = {Sl[0] * iD, Sl[1] * iD, Sl[2] * iD};
  const double Bs[3] = {B[0] * isD, B[1] * isD, B[2] * isD};
  double ru[3], Bsl[3];
  sym_apply(gu, rl, ru);
  sym_apply(gl, Bs, Bsl);
  s.ye = fmax(fmin(ye, par.ye_max), par.ye_min);
  if (KIND == 2) {
    s.tab.hint = -1; s.tab.cell.ir = -1;
    s.tab.lrho.x = s.tab.leps.x = 0.0; s.tab.lrho.ix = s.tab.leps.ix = INFINITY;        // empty references: the range test fails,
    s.tab.lrho.l = s.tab.leps.l = 0.0; s.tab.lp.l = 1e300; s.tab.lp.p = 0.0;            // the first evaluation sets them
    s.ypos = tab_locate(s.ye, par.ye0, par.idye, par.n_ye);
  }
  s.r2 = ru[0] * rl[0] + ru[1] * rl[1] + ru[2] * rl[2];                            // (D2)
  s.B2 = Bs[0] * Bsl[0] + Bs[1] * Bsl[1] + Bs[2] * Bsl[2];
  const double rB = rl[0] * Bs[0] + rl[1] * Bs[1] + rl[2] * Bs[2];
  s.rB2 = rB * rB;
  s.B2rp2 = s.B2 * s.r2 - s.rB2;
  s.h0 = KIND == 2 ? par.tab_h0 : 1.0;
  s.v02 = s.r2 / (s.h0 * s.h0 + s.r2);
  if (KIND == 2) { s.rho_lo = par.tab_rho_lo; s.rho_hi = par.tab_rho_hi; }
  else { s.rho_lo = 0.0; s.rho_hi = par.rho_max; }
  const double mub = 1.0 / s.h0;
  // ---- the two root solves of App. D (steps 2-3), written as ONE loop with ONE evaluation site of the master function f, so
  // that all lanes of a warp run the same instructions whatever stage of the solve they are in and the (long) body of f exists
  // once in the instruction stream. Stages:
  //   WARM_A, WARM_B  warm start: the primitive slot still holds the solution of the previous stage, which for a time-stepped
  //                   state lies within ~1e-3 of the new one. mu0 = 1 / (W h) of it and a second point one doubled Newton step
  //                   away (f' ~ 1: f = mu - 1 / (nu + mu rbar^2), nu varies slowly; the doubled step overshoots the root) are
  //                   used as the bracket of step 3 if f changes sign between them (the root of f on (0, mu_+] is unique and f
  //                   grows beyond mu_+); otherwise
  //   COLD_0, COLD_1  steps 2-3 as printed: mu_+ from f_a (D3), then f(0), f(mu_+) (R9: degenerate root at the bracket end);
  //   BRENT           Brent's bracketing iteration (l.1143), to 2 ulp of mu or c2p_maxit evaluations;
  //   FINAL           one more evaluation if the accepted end of the bracket is not the point evaluated last (the primitives
  //                   are by-products of the evaluation at the root: step 4).
  // The result is the same root to the tolerance of the solver whichever way the bracket was found.
  enum { WARM_A, WARM_B, COLD_0, COLD_1, BRENT, FINAL };
  bool ok1 = true, ok2 = true;
  double mu = 0.0, mu_plus = 0.0, f0 = 0.0;
  double ba = 0.0, fa = 0.0, bb = 0.0, fb = 0.0, bc = 0.0, fc = 0.0, bd = 0.0, be = 0.0;   // Brent: a, b (best), c (other end), last two steps
  int state, it = 0;
  double xe;                                                                      // point to evaluate next
  auto solve_mu_plus = [&]() { return brent_root([&](double m) { return s.fa(m); }, 0.0, mub, -1.0, s.fa(mub), par.c2p_maxit, ok1); };   // step 2
  {
    const double Wo = P[(size_t)WLOR * sp + pt], ro = P[(size_t)RHO * sp + pt], eo = P[(size_t)EPS * sp + pt], po = P[(size_t)PRESS * sp + pt];
    const double mu0 = ro / (Wo * (ro * (1.0 + eo) + po));
    if (mu0 > 0.0 && mu0 < mub) {                      // false for NaN / zero-initialised primitives
      if (KIND == 2) {                                 // the old temperature points at the table cell to try first
        const double To = P[(size_t)TEMP * sp + pt];
        if (To > 0.0) s.tab.hint = tab_locate((double)(__log2f((float)To) * 0.30103f), par.lT0, par.idlT, par.n_T).i;   // a hint only: single precision will do
      }
      state = WARM_A; xe = mu0;
    } else { mu_plus = solve_mu_plus(); state = COLD_0; xe = 0.0; }
  }
  for (;;) {
    const double fx = s.f(par, xe);
    if (state == FINAL) { mu = xe; break; }
    if (state == WARM_A) {
      const double xb = fmin(fmax(xe - 2.0 * fx, 0.5 * xe), mub);
      if (fx == 0.0 || xb == xe) { mu = xe; break; }  // the step is below one ulp: mu0 is the root to solver tolerance
      ba = xe; fa = fx; xe = xb; state = WARM_B;
      continue;
    }
    if (state == COLD_0) { f0 = fx; xe = mu_plus; state = COLD_1; continue; }
    if (state == WARM_B) {
      if ((fa < 0.0) == (fx < 0.0)) { mu_plus = solve_mu_plus(); state = COLD_0; xe = 0.0; continue; }   // no bracket: start cold
      bb = xe; fb = fx;
    } else if (state == COLD_1) {
      if ((f0 > 0.0) == (fx > 0.0) && fx != 0.0 && f0 != 0.0) { mu = xe; ok2 = fabs(fx) <= 1e-12; break; }   // R9: degenerate root at the bracket end
      ba = 0.0; fa = f0; bb = xe; fb = fx;
    } else fb = fx;                                    // BRENT: bb == xe
    if (state != BRENT) { bc = ba; fc = fa; bd = bb - ba; be = bd; it = 0; state = BRENT; }
    // ---- one step of Brent's method: bracket [bb, bc], bb the better end
    if ((fb > 0.0) == (fc > 0.0)) { bc = ba; fc = fa; bd = bb - ba; be = bd; }
    if (fabs(fc) < fabs(fb)) { ba = bb; bb = bc; bc = ba; fa = fb; fb = fc; fc = fa; }
    const double tol = 2.0 * DBL_EPSILON * fabs(bb);
    const double m = 0.5 * (bc - bb);
    bool done = fabs(m) <= tol || fb == 0.0;
    if (!done && it >= par.c2p_maxit) { ok2 = false; done = true; }
    if (done) {
      if (bb == xe) { mu = bb; break; }
      xe = bb; state = FINAL;
      continue;
    }
    ++it;
    if (fabs(be) < tol || fabs(fa) <= fabs(fb)) { bd = m; be = m; }
    else {
      double pp, qq, rr, ss = fb / fa;
      if (ba == bc) { pp = 2.0 * m * ss; qq = 1.0 - ss; }
      else { qq = fa / fc; rr = fb / fc; pp = ss * (2.0 * m * qq * (qq - rr) - (bb - ba) * (rr - 1.0)); qq = (qq - 1.0) * (rr - 1.0) * (ss - 1.0); }
      if (pp > 0.0) qq = -qq; else pp = -pp;
      ss = be; be = bd;
      if (2.0 * pp < 3.0 * m * qq - fabs(tol * qq) && pp < fabs(0.5 * ss * qq)) bd = pp / qq;
      else { bd = m; be = m; }
    }
    ba = bb; fa = fb;
    bb += fabs(bd) > tol ? bd : (m > 0.0 ? tol : -tol);
    xe = bb;
  }
  if (!ok1 || !ok2) flag |= MHD_FLAG_NOCONV;
  W = s.W; rho = D / W; eps = s.eps_raw;
  const double x = s.x_of(mu);
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] = mu * x * (ru[i] + mu * rB * Bs[i]);           // (D15)
  // ---- error policy
  if (!(rho >= par.rho_cut)) { store_atmosphere(io, par, pt, atmo, flag); return; }    // rule 1
  const bool allowed = (rho < par.rho_low) || bh;
  if (rho > par.rho_max) flag |= MHD_FLAG_FATAL;                                   // rule 2
  if (KIND == 2) {
    // rules 3-4 with the table: "eps outside [eps_min, eps_max](rho, Ye)" is the clamp the last evaluation of f (at the root) applied
    // itself (same rho, same columns, compared in log space); an evaluation that found eps inside a table cell is inside the range
    if (s.tab.clamp != 0) {
      const double rho_c = fmax(fmin(s.rho_hi, rho), s.rho_lo);
      const TPos r = tab_locate(log10_1(rho_c), par.lr0, par.idlr, par.n_rho);
      eps = exp10_1(tab_ecol(par, r, s.ypos, s.tab.clamp < 0 ? 0 : par.n_T - 1)) - par.tab_eps_shift;
      changed = true;
      if (s.tab.clamp < 0) flag |= MHD_FLAG_EPS_LO;                                // rule 3
      else flag |= allowed ? MHD_FLAG_EPS_HI : (MHD_FLAG_EPS_HI | MHD_FLAG_FATAL); // rule 4
    }
  } else {
    double emin, emax;
    eos_eps_range<KIND>(par, fmax(fmin(s.rho_hi, rho), s.rho_lo), s.ye, emin, emax);
    if (eps < emin) { eps = emin; flag |= MHD_FLAG_EPS_LO; changed = true; }       // rule 3
    else if (eps > emax) { eps = emax; changed = true; flag |= allowed ? MHD_FLAG_EPS_HI : (MHD_FLAG_EPS_HI | MHD_FLAG_FATAL); }   // rule 4
  }
  if (W > par.w_max) {                                                             // rule 5
    flag |= allowed ? MHD_FLAG_VMAX : (MHD_FLAG_VMAX | MHD_FLAG_FATAL);
    const double vmax2 = 1.0 - 1.0 / (par.w_max * par.w_max);
    double vl[3];
    sym_apply(gl, v, vl);
    const double v2 = v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2];
    const double sc = sqrt(vmax2 / v2);
    v[0] *= sc; v[1] *= sc; v[2] *= sc;
    W = par.w_max; rho = D / W; changed = true;
  }
  if (ye < par.ye_min || ye > par.ye_max) {                                        // rule 6
    flag |= allowed ? MHD_FLAG_YE : (MHD_FLAG_YE | MHD_FLAG_FATAL);
    ye = par.ye_atmo; changed = true;
  }
  Eos e;
  if (KIND == 2 && !changed) {
    // no rule acted: (rho, eps, Ye) are those of the last evaluation of f, whose table position is still at hand
    e.p = s.p_last;
    e.T = exp10_1(par.lT0 + ((double)s.tab.tpos.i + s.tab.tpos.w) * par.dlT);
    e.cs2 = tab_tri(par, par.tab_cs2, s.tab.rpos, s.tab.tpos, s.ypos);
  } else e = eos_eval<KIND>(par, rho, eps, ye);
  store_point(io, pt, gl, sg, B, rho, ye, eps, e, v, W, flag, changed);
}

// The inputs of a cell that is going to be solved are pulled into L1 ahead of time: the solve is hundreds of dependent instructions at four CTAs per SM,
// nothing else covers the latency of its 20 input loads (D and chi were read by pass A)
template <int KIND>
__device__ __forceinline__ void prefetch_inputs(const double* U, size_t su, const double* P, size_t sp, size_t q) {
  auto pf = [](const double* a) { asm volatile("prefetch.global.L1 [%0];" ::"l"(a)); };
#pragma unroll
  for (int f = 0; f < 6; ++f) pf(U + (size_t)(GXX + f) * su + q);
  pf(U + (size_t)ALPHA * su + q);
#pragma unroll
  for (int f = 0; f < 8; ++f) pf(U + (size_t)(DYEBAR + f) * su + q);   // DYe, tau, S_i, B^i
  pf(P + (size_t)WLOR * sp + q); pf(P + (size_t)RHO * sp + q); pf(P + (size_t)EPS * sp + q); pf(P + (size_t)PRESS * sp + q);
  if (KIND == 2) pf(P + (size_t)TEMP * sp + q);
}

template <int KIND>
__global__ void __launch_bounds__(C2P_THREADS, 4) k_con2prim(const __grid_constant__ Dims d, const __grid_constant__ Par par,
                                                             double* __restrict__ U, size_t su, double* __restrict__ P, size_t sp,
                                                             uint8_t* __restrict__ flags, const double* __restrict__ atmo) {
  __shared__ int list[C2P_CHUNK];
  __shared__ int count;
  const C2pIo io = {U, su, P, sp, flags};
  const int tid = threadIdx.x, lane = tid & 31;
  if (tid == 0) count = 0;
  __syncthreads();
  const long long chunk0 = (long long)blockIdx.x * C2P_CHUNK;
  // ---- pass A: atmosphere pre-check (note N2), atmosphere cells written at once, the others compacted
#pragma unroll
  for (int r = 0; r < C2P_PER_THREAD; ++r) {
    const long long pt = chunk0 + r * C2P_THREADS + tid;
    bool solve = false;
    if (pt < d.npts) {
      const double chi = U[(size_t)CHI * su + pt];
      const double D = U[(size_t)DBAR * su + pt] * (chi * sqrt(chi));
      solve = D >= par.rho_cut;                                                    // false for NaN as well
      if (!solve) store_atmosphere(io, par, pt, atmo, 0u);
    }
    const unsigned b = __ballot_sync(0xffffffffu, solve);
    int base = 0;
    if (lane == 0 && b) base = atomicAdd(&count, __popc(b));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (solve) {
      const int pos = base + __popc(b & ((1u << lane) - 1u));
      list[pos] = (int)(pt - chunk0);
      if (pos < C2P_THREADS) prefetch_inputs<KIND>(U, su, P, sp, (size_t)pt);   // the first cell of each thread of pass B
    }
  }
  __syncthreads();
  // ---- pass B: the solve, dense
  const int n = count;
  for (int e = tid; e < n; e += C2P_THREADS) {
    if (e + C2P_THREADS < n) prefetch_inputs<KIND>(U, su, P, sp, (size_t)(chunk0 + list[e + C2P_THREADS]));   // this thread's next cell, while this one is solved
    solve_point<KIND>(io, par, chunk0 + list[e], atmo);
  }
}

template <int KIND>
__global__ void __launch_bounds__(128) k_prim2con(const __grid_constant__ Dims d, const __grid_constant__ Par par,
                                                  double* __restrict__ U, size_t su, double* __restrict__ P, size_t sp) {
  const long long pt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (pt >= d.npts) return;
  auto u = [&](int f) -> double& { return U[(size_t)f * su + pt]; };
  auto pr = [&](int f) -> double& { return P[(size_t)f * sp + pt]; };
  const double chi = u(CHI);
  const double isg = chi * sqrt(chi), sg = 1.0 / isg;
  const Sym3 gt = {u(GXX), u(GXY), u(GXZ), u(GYY), u(GYZ), u(GZZ)};
  const Sym3 gl = sym_scale(gt, 1.0 / chi);
  const double rho = pr(RHO), eps = pr(EPS), ye = pr(YE);
  const double v[3] = {pr(VX), pr(VY), pr(VZ)};
  const double B[3] = {u(BXBAR) * isg, u(BYBAR) * isg, u(BZBAR) * isg};
  const Eos e = eos_eval<KIND>(par, rho, eps, ye);
  double D, tau, S[3], W;
  cons_from_prim(gl, rho, eps, e.p, v, B, D, tau, S, W);
  pr(PRESS) = e.p; pr(TEMP) = e.T; pr(CS2) = e.cs2; pr(WLOR) = W;
  u(DBAR) = sg * D; u(DYEBAR) = sg * D * ye; u(TAUBAR) = sg * tau;
  u(SXBAR) = sg * S[0]; u(SYBAR) = sg * S[1]; u(SZBAR) = sg * S[2];
}

cudaError_t launch_con2prim(const Dims& d, const Par& par, double* U, size_t su, double* P, size_t sp, uint8_t* flags, double* atmo, cudaStream_t s) {
  const unsigned nb = (unsigned)((d.npts + C2P_CHUNK - 1) / C2P_CHUNK);
  if (par.eos_kind == 0) { k_atmo_state<0><<<1, 32, 0, s>>>(par, atmo); k_con2prim<0><<<nb, C2P_THREADS, 0, s>>>(d, par, U, su, P, sp, flags, atmo); }
  else if (par.eos_kind == 1) { k_atmo_state<1><<<1, 32, 0, s>>>(par, atmo); k_con2prim<1><<<nb, C2P_THREADS, 0, s>>>(d, par, U, su, P, sp, flags, atmo); }
  else { k_atmo_state<2><<<1, 32, 0, s>>>(par, atmo); k_con2prim<2><<<nb, C2P_THREADS, 0, s>>>(d, par, U, su, P, sp, flags, atmo); }
  return cudaGetLastError();
}
cudaError_t launch_prim2con(const Dims& d, const Par& par, double* U, size_t su, double* P, size_t sp, cudaStream_t s) {
  const unsigned nb = (unsigned)((d.npts + 127) / 128);
  if (par.eos_kind == 0) k_prim2con<0><<<nb, 128, 0, s>>>(d, par, U, su, P, sp);
  else if (par.eos_kind == 1) k_prim2con<1><<<nb, 128, 0, s>>>(d, par, U, su, P, sp);
  else k_prim2con<2><<<nb, 128, 0, s>>>(d, par, U, su, P, sp);
  return cudaGetLastError();
}

}  // namespace mhd
