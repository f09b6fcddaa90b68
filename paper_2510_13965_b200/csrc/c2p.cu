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
// One thread per grid point; x-contiguous warps so the 18 loads and 11 stores per point coalesce.
// Divergence control: atmosphere cells skip the solve entirely; both root solves are bounded by c2p_maxit.
#include <float.h>
#include "mhd_internal.cuh"
#include "rootfind.cuh"

namespace mhd {

// ------------------------------------------------------------------------------------------ EoS
struct Eos { double p, T, cs2; };

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
__device__ __forceinline__ TPos tab_locate(double x, double x0, double dx, int n) {
  double s = (x - x0) / dx;
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
    const TPos r = tab_locate(log10(rho), q.lr0, q.dlr, q.n_rho);
    const TPos y = tab_locate(ye, q.ye0, q.dye, q.n_ye);
    const TPos t = tab_T_of_loge(q, r, y, log10(eps + q.tab_eps_shift));
    o.p = exp10(tab_tri(q, q.tab_logp, r, t, y));
    o.T = exp10(q.lT0 + ((double)t.i + t.w) * q.dlT);
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
    const TPos r = tab_locate(log10(rho), q.lr0, q.dlr, q.n_rho);
    const TPos y = tab_locate(ye, q.ye0, q.dye, q.n_ye);
    emin = exp10(tab_col(q, q.tab_loge, r, y, 0)) - q.tab_eps_shift;
    emax = exp10(tab_col(q, q.tab_loge, r, y, q.n_T - 1)) - q.tab_eps_shift;
  }
}
__device__ __forceinline__ double eos_eps_of_T(const Par& q, double rho, double T, double ye) {
  const TPos r = tab_locate(log10(rho), q.lr0, q.dlr, q.n_rho);
  const TPos y = tab_locate(ye, q.ye0, q.dye, q.n_ye);
  const TPos t = tab_locate(log10(T), q.lT0, q.dlT, q.n_T);
  return exp10(tab_tri(q, q.tab_loge, r, t, y)) - q.tab_eps_shift;
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
// State of the App. D master function; one instance per thread.
// Tabulated EoS inside the mu iteration: pressure and clamped eps for (rho, eps_raw) at fixed Ye. Same interpolant and
// same clamps as eos_eps_range + eos_eval, arranged for the iteration: one log10 per argument, the eps range compared in
// log space (no pow unless the clamp acts), T and cs2 not evaluated, and the T cell of the previous evaluation tried
// first (the interpolant is monotone along T, so whatever the search order the cell found is the same).
__device__ __forceinline__ void tab_p_of_eps(const Par& q, TPos y, double rho, double eps_raw, int& hint, double& p, double& eps) {
  const TPos r = tab_locate(log10(rho), q.lr0, q.dlr, q.n_rho);
  const double e_min = tab_col(q, q.tab_loge, r, y, 0), e_max = tab_col(q, q.tab_loge, r, y, q.n_T - 1);
  const double le = log10(eps_raw + q.tab_eps_shift);
  TPos t;
  if (!(le > e_min)) { t.i = 0; t.w = 0.0; eps = exp10(e_min) - q.tab_eps_shift; }
  else if (le >= e_max) { t.i = q.n_T - 2; t.w = 1.0; eps = exp10(e_max) - q.tab_eps_shift; }
  else {
    eps = eps_raw;
    int lo = 0, hi = q.n_T - 1;
    double e_lo = e_min, e_hi = e_max;
    if (hint >= 0 && hint < q.n_T - 1) {               // the cell of the last evaluation, then its neighbours, then bisection
      const double a = tab_col(q, q.tab_loge, r, y, hint), b = tab_col(q, q.tab_loge, r, y, hint + 1);
      if (le >= a) { lo = hint; e_lo = a; if (le < b) { hi = hint + 1; e_hi = b; } else { lo = hint + 1; e_lo = b; } }
      else { hi = hint; e_hi = a; }
    }
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      const double em = tab_col(q, q.tab_loge, r, y, mid);
      if (le >= em) { lo = mid; e_lo = em; } else { hi = mid; e_hi = em; }
    }
    t.i = lo; t.w = (le - e_lo) / (e_hi - e_lo);
    hint = lo;
  }
  p = exp10(tab_tri(q, q.tab_logp, r, t, y));
}

template <int KIND>
struct Master {
  double D, q, r2, B2, rB2, B2rp2, ye, h0, v02, rho_lo, rho_hi;
  double W, eps_raw;   // by-products of the last evaluation
  TPos ypos;           // table position of Ye (fixed during the solve)
  int t_hint;          // T cell of the last table evaluation
  __device__ __forceinline__ double x_of(double mu) const { return 1.0 / (1.0 + mu * B2); }          // (D5)
  __device__ __forceinline__ double rbar2(double mu) const {                                          // (D4)
    const double x = x_of(mu);
    return r2 * x * x + mu * x * (1.0 + x) * rB2;
  }
  __device__ __forceinline__ double fa(double mu) const { return mu * sqrt(h0 * h0 + rbar2(mu)) - 1.0; }   // (D3)
  __device__ __forceinline__ double f_body(const Par& par, double mu) {                                   // (D6)-(D14)
    const double x = x_of(mu);
    const double rb2 = rbar2(mu);
    const double qbar = q - 0.5 * B2 - 0.5 * mu * mu * x * x * B2rp2;
    const double v2 = fmin(mu * mu * rb2, v02);
    const double iW = sqrt(1.0 - v2);
    W = 1.0 / iW;
    double rho = D * iW;
    rho = fmax(fmin(rho_hi, rho), rho_lo);
    eps_raw = W * ((qbar - mu * rb2) + v2 / (1.0 + iW));                                             // (D12): W^2/(1+W) = W/(1+1/W)
    double eps, p;
    if (KIND == 2) tab_p_of_eps(par, ypos, rho, eps_raw, t_hint, p, eps);
    else {
      double emin, emax;
      eos_eps_range<KIND>(par, rho, ye, emin, emax);
      eps = fmax(fmin(emax, eps_raw), emin);
      p = eos_eval<KIND>(par, rho, eps, ye).p;
    }
    const double a = p / (rho * (1.0 + eps));
    const double nuA = (1.0 + a) * (1.0 + eps) * iW;
    const double nuB = (1.0 + a) * (1.0 + qbar - mu * rb2);
    return mu - 1.0 / (fmax(nuA, nuB) + mu * rb2);
  }
  // the table version is evaluated from seven places and is ~700 instructions long: one out-of-line copy keeps the kernel
  // inside the instruction cache (its top stall was no_instruction); the analytic EoS versions are short and stay inline
  __device__ __noinline__ double f_out(const Par& par, double mu) { return f_body(par, mu); }
  __device__ __forceinline__ double f(const Par& par, double mu) { return KIND == 2 ? f_out(par, mu) : f_body(par, mu); }
};

// ------------------------------------------------------------------------------------------ kernels
template <int KIND>
__global__ void __launch_bounds__(128, 4) k_con2prim(const __grid_constant__ Dims d, const __grid_constant__ Par par,
                                                  double* __restrict__ U, size_t su, double* __restrict__ P, size_t sp,
                                                  uint8_t* __restrict__ flags) {
  const long long pt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (pt >= d.npts) return;
  auto u = [&](int f) -> double& { return U[(size_t)f * su + pt]; };
  Sym3 gt = {u(GXX), u(GXY), u(GXZ), u(GYY), u(GYZ), u(GZZ)};
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
  double rho = 0.0, eps = 0.0, W = 1.0, v[3] = {0.0, 0.0, 0.0};
  bool atmo = !(D >= par.rho_cut), changed = false;
  const bool bh = alpha < par.alpha_bh;

  if (!atmo) {
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
    s.t_hint = -1;
    if (KIND == 2) s.ypos = tab_locate(s.ye, par.ye0, par.dye, par.n_ye);
    s.r2 = ru[0] * rl[0] + ru[1] * rl[1] + ru[2] * rl[2];                            // (D2)
    s.B2 = Bs[0] * Bsl[0] + Bs[1] * Bsl[1] + Bs[2] * Bsl[2];
    const double rB = rl[0] * Bs[0] + rl[1] * Bs[1] + rl[2] * Bs[2];
    s.rB2 = rB * rB;
    s.B2rp2 = s.B2 * s.r2 - s.rB2;
    s.h0 = KIND == 2 ? par.tab_h0 : 1.0;
    s.v02 = s.r2 / (s.h0 * s.h0 + s.r2);
    if (KIND == 2) { s.rho_lo = exp10(par.lr0); s.rho_hi = exp10(par.lr0 + par.dlr * (par.n_rho - 1)); }
    else { s.rho_lo = 0.0; s.rho_hi = par.rho_max; }
    bool ok1 = true, ok2 = true;
    const double mub = 1.0 / s.h0;
    double mu = 0.0;
    // Warm start: the primitive slot still holds the solution of the previous stage, which for a time-stepped state lies
    // within ~1e-3 of the new one. mu0 = 1 / (W h) of it and a second point one doubled Newton step away are tried as the
    // bracket of step 3; they are used only if f changes sign between them (the root of f on (0, mu_+] is unique, and f grows beyond mu_+), otherwise the solve starts cold
    // from steps 2-3 as printed. The result is the same root to the tolerance of the solver either way.
    bool warm = false;
    {
      const double Wo = P[(size_t)WLOR * sp + pt], ro = P[(size_t)RHO * sp + pt], eo = P[(size_t)EPS * sp + pt], po = P[(size_t)PRESS * sp + pt];
      const double mu0 = ro / (Wo * (ro * (1.0 + eo) + po));
      if (mu0 > 0.0 && mu0 < mub) {                      // false for NaN / zero-initialised primitives
        // second point by a doubled Newton step with f' ~ 1 (f = mu - 1 / (nu + mu rbar^2), nu varies slowly): it
        // overshoots the root, so the two points bracket it with a width of ~2 |f(mu0)|
        const double fa_ = s.f(par, mu0);
        const double b = fmin(fmax(mu0 - 2.0 * fa_, 0.5 * mu0), mub);
        const bool hit = fa_ == 0.0 || b == mu0;        // the step is below one ulp: mu0 is the root to solver tolerance
        const double fb_ = hit ? 0.0 : s.f(par, b);
        if (hit) { mu = mu0; warm = true; }
        else if ((fa_ < 0.0) != (fb_ < 0.0)) {
          mu = brent_root([&](double m) { return s.f(par, m); }, mu0, b, fa_, fb_, par.c2p_maxit, ok2);
          warm = true;
        }
      }
    }
    if (!warm) {
      const double mu_plus = brent_root([&](double m) { return s.fa(m); }, 0.0, mub, -1.0, s.fa(mub), par.c2p_maxit, ok1);   // step 2
      const double f0 = s.f(par, 0.0), f1 = s.f(par, mu_plus);
      if ((f0 > 0.0) == (f1 > 0.0) && f1 != 0.0 && f0 != 0.0) { mu = mu_plus; ok2 = fabs(f1) <= 1e-12; }   // R9: degenerate root at the bracket end
      else mu = brent_root([&](double m) { return s.f(par, m); }, 0.0, mu_plus, f0, f1, par.c2p_maxit, ok2);                 // step 3
    }
    s.f(par, mu);                                                                    // step 4
    if (!ok1 || !ok2) flag |= MHD_FLAG_NOCONV;
    W = s.W; rho = D / W; eps = s.eps_raw;
    const double x = s.x_of(mu);
#pragma unroll
    for (int i = 0; i < 3; ++i) v[i] = mu * x * (ru[i] + mu * rB * Bs[i]);           // (D15)
    // ---- error policy
    if (!(rho >= par.rho_cut)) atmo = true;                                          // rule 1
    else {
      const bool allowed = (rho < par.rho_low) || bh;
      if (rho > par.rho_max) flag |= MHD_FLAG_FATAL;                                 // rule 2
      double emin, emax;
      eos_eps_range<KIND>(par, fmax(fmin(s.rho_hi, rho), s.rho_lo), s.ye, emin, emax);
      if (eps < emin) { eps = emin; flag |= MHD_FLAG_EPS_LO; changed = true; }       // rule 3
      else if (eps > emax) { eps = emax; changed = true; flag |= allowed ? MHD_FLAG_EPS_HI : (MHD_FLAG_EPS_HI | MHD_FLAG_FATAL); }   // rule 4
      if (W > par.w_max) {                                                           // rule 5
        flag |= allowed ? MHD_FLAG_VMAX : (MHD_FLAG_VMAX | MHD_FLAG_FATAL);
        const double vmax2 = 1.0 - 1.0 / (par.w_max * par.w_max);
        double vl[3];
        sym_apply(gl, v, vl);
        const double v2 = v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2];
        const double sc = sqrt(vmax2 / v2);
        v[0] *= sc; v[1] *= sc; v[2] *= sc;
        W = par.w_max; rho = D / W; changed = true;
      }
      if (ye < par.ye_min || ye > par.ye_max) {                                      // rule 6
        flag |= allowed ? MHD_FLAG_YE : (MHD_FLAG_YE | MHD_FLAG_FATAL);
        ye = par.ye_atmo; changed = true;
      }
    }
  }
  if (atmo) {
    flag |= MHD_FLAG_ATMO;
    rho = par.rho_atmo; W = 1.0; v[0] = v[1] = v[2] = 0.0; ye = par.ye_atmo;
    if (KIND == 2) eps = eos_eps_of_T(par, rho, par.T_atmo, ye);
    else if (KIND == 1) { double emin, emax; eos_eps_range<KIND>(par, rho, ye, emin, emax); eps = emin + par.eps_atmo; }
    else eps = par.eps_atmo;
    changed = true;
  }
  const Eos e = eos_eval<KIND>(par, rho, eps, ye);
  P[(size_t)RHO * sp + pt] = rho; P[(size_t)YE * sp + pt] = ye; P[(size_t)EPS * sp + pt] = eps; P[(size_t)PRESS * sp + pt] = e.p;
  P[(size_t)VX * sp + pt] = v[0]; P[(size_t)VY * sp + pt] = v[1]; P[(size_t)VZ * sp + pt] = v[2];
  P[(size_t)WLOR * sp + pt] = W; P[(size_t)TEMP * sp + pt] = e.T; P[(size_t)CS2 * sp + pt] = e.cs2;
  flags[pt] = (uint8_t)flag;
  if (changed) {                                                                     // R11
    double Dn, taun, Sn[3], Wn;
    cons_from_prim(gl, rho, eps, e.p, v, B, Dn, taun, Sn, Wn);
    u(DBAR) = sg * Dn; u(DYEBAR) = sg * Dn * ye; u(TAUBAR) = sg * taun;
    u(SXBAR) = sg * Sn[0]; u(SYBAR) = sg * Sn[1]; u(SZBAR) = sg * Sn[2];
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

cudaError_t launch_con2prim(const Dims& d, const Par& par, double* U, size_t su, double* P, size_t sp, uint8_t* flags, cudaStream_t s) {
  const unsigned nb = (unsigned)((d.npts + 127) / 128);
  if (par.eos_kind == 0) k_con2prim<0><<<nb, 128, 0, s>>>(d, par, U, su, P, sp, flags);
  else if (par.eos_kind == 1) k_con2prim<1><<<nb, 128, 0, s>>>(d, par, U, su, P, sp, flags);
  else k_con2prim<2><<<nb, 128, 0, s>>>(d, par, U, su, P, sp, flags);
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
