// LES gradient sub-grid-scale tensors: PAPER.md Sec. II B l.252-256 and App. A, Eqs. (A11)-(A17) l.855-882.
// The induction equation's, coefficient C_M (the paper's production setting: C_M = 8, the other coefficients 0, l.863), is the default
// instantiation; with any of C_N, C_Y, C_T set the FULL instantiations add H_N^k, H_{N_Y}^k (A15) and H_T^{ki} (A17) to the fluxes of Dbar, DYebar, Sbar_i.
//   -alpha G_B^{ki} = +alpha C_M xi sqrt(gamma) H_M^{ki},   xi = gamma^{1/3} Delta^2 / 24,
// is part of the flux bracket of Bbar^i in direction k (Eq. 32): it is ADDED to the pointwise fluxes of the work slot after
// k_point_flux and before the flux-splitting reconstruction. Readings of the appendix's undefined symbols: DESIGN.md R39-R44
// (calE = h W^2 with the enthalpy density h, Theta = calE + B^2, E^i = -eps^{ijk} v_j B_k; first index of H_M = flux direction).
// Two streaming kernels:
//   k_les_aux    every grid point: the 26 scalar fields whose gradients App. A contracts (B^k, v^k, v_k, B_k, E_k, E^k, v.B, Theta,
//                W^-2, rho, eps, h, dp/drho, dp/deps) -> MHD_SLOT_LESWORK
//   k_les_flux   every grid point at least 2 points inside the array: fourth-order centred gradients (Eq. 60) of those fields, the 36
//                products grad f . grad g = gamma^{mn} d_m f d_n g that (A12)-(A16) need, then the closed forms; bound by L1/L2 loads
//                (26 fields x 12 neighbours per point).
// EoS derivatives: analytic for the ideal gas and the hybrid piecewise polytrope (l.882); derivatives of the interpolant in the cell for the table (R42).
#include "mhd_internal.cuh"
#include "tma.cuh"
#include <utility>

namespace mhd {

namespace {

enum { A_BU = 0, A_VU = 3, A_VL = 6, A_BL = 9, A_EL = 12, A_EU = 15, A_VB = 18, A_TH = 19, A_WM2 = 20, A_RHO = 21, A_EPS = 22, A_H = 23,
       A_DPR = 24, A_DPE = 25, A_YE = 26, A_DPY = 27, A_D = 28, A_CALE = 29, A_DYE = 30, NAUX = MHD_NLESWORK, NAUX_NOYE = 26 };
// Ye, dp/dYe only with the tabulated EoS; D with it or with FULL; calE, D Ye only with FULL (any of C_N, C_Y, C_T set: (A15), (A17))
static_assert(NAUX == 31, "MHD_NLESWORK and the field list disagree");
__host__ __device__ constexpr int sym3(int i, int j) { return i == j ? (i == 0 ? 0 : i == 1 ? 3 : 5) : (i + j == 1 ? 1 : i + j == 2 ? 2 : 4); }

// ---- tabulated EoS: derivatives of the trilinear interpolant inside the cell that holds (rho, T, Ye) (reading R42)
struct TabCell { int ir, it, iy; double wr, wt, wy; };
__device__ __forceinline__ void tab_pos(double x, double x0, double idx, int n, int& i, double& w) {
  double s = fmin(fmax((x - x0) * idx, 0.0), (double)(n - 1));
  i = min((int)s, n - 2);
  w = s - (double)i;
}
// value of table t at T node `it`, bilinear in (log10 rho, Ye)
__device__ __forceinline__ double tab_column(const Par& q, const double* __restrict__ t, const TabCell& c, int it) {
  const size_t b0 = ((size_t)c.iy * q.n_T + it) * q.n_rho + c.ir, b1 = b0 + (size_t)q.n_T * q.n_rho;
  const double lo = __ldg(t + b0) + c.wr * (__ldg(t + b0 + 1) - __ldg(t + b0)), hi = __ldg(t + b1) + c.wr * (__ldg(t + b1 + 1) - __ldg(t + b1));
  return lo + c.wy * (hi - lo);
}
__device__ __noinline__ void table_dp(const Par& q, double rho, double eps, double ye, double& dpr, double& dpe, double& dpy) {
  TabCell c;
  tab_pos(log10(rho), q.lr0, q.idlr, q.n_rho, c.ir, c.wr);
  tab_pos(ye, q.ye0, q.idye, q.n_ye, c.iy, c.wy);
  const double le = log10(eps + q.tab_eps_shift);
  {                                                          // T by inversion of the interpolant along the monotone log T axis, clamped
    int lo = 0, hi = q.n_T - 1;
    double e_lo = tab_column(q, q.tab_loge, c, lo), e_hi = tab_column(q, q.tab_loge, c, hi);
    if (le <= e_lo) { c.it = 0; c.wt = 0.0; }
    else if (le >= e_hi) { c.it = q.n_T - 2; c.wt = 1.0; }
    else {
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        const double em = tab_column(q, q.tab_loge, c, mid);
        if (le >= em) { lo = mid; e_lo = em; } else { hi = mid; e_hi = em; }
      }
      c.it = lo; c.wt = (le - e_lo) / (e_hi - e_lo);
    }
  }
  // the 8 corners of both tables; slope along an axis = difference of the two faces across it (each bilinear in the other two) / spacing
  double sl[2][3], val = 0.0;
#pragma unroll
  for (int tb = 0; tb < 2; ++tb) {
    const double* __restrict__ t = tb == 0 ? q.tab_logp : q.tab_loge;
    double v[2][2][2];                                       // [rho][T][Ye]
#pragma unroll
    for (int cy = 0; cy < 2; ++cy)
#pragma unroll
      for (int ct = 0; ct < 2; ++ct) {
        const size_t b = ((size_t)(c.iy + cy) * q.n_T + (c.it + ct)) * q.n_rho + c.ir;
        v[0][ct][cy] = __ldg(t + b); v[1][ct][cy] = __ldg(t + b + 1);
      }
    const double wr[2] = {1.0 - c.wr, c.wr}, wt[2] = {1.0 - c.wt, c.wt}, wy[2] = {1.0 - c.wy, c.wy};
    double sr = 0.0, st = 0.0, sy = 0.0, s0 = 0.0;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        sr += wt[a] * wy[b] * (v[1][a][b] - v[0][a][b]);
        st += wr[a] * wy[b] * (v[a][1][b] - v[a][0][b]);
        sy += wr[a] * wt[b] * (v[a][b][1] - v[a][b][0]);
#pragma unroll
        for (int e = 0; e < 2; ++e) s0 += wr[a] * wt[b] * wy[e] * v[a][b][e];
      }
    sl[tb][0] = sr * q.idlr; sl[tb][1] = st * q.idlT; sl[tb][2] = sy * q.idye;
    if (tb == 0) val = s0;
  }
  const double p = exp10(val);
  dpr = p / rho * (sl[0][0] - sl[0][1] * sl[1][0] / sl[1][1]);
  dpe = p / (eps + q.tab_eps_shift) * (sl[0][1] / sl[1][1]);
  dpy = p * 2.302585092994045684 * (sl[0][2] - sl[0][1] * sl[1][2] / sl[1][1]);
}


template <bool TABLE, bool FULL>
__global__ void __launch_bounds__(128) k_les_aux(const __grid_constant__ Dims d, const __grid_constant__ Par par, const double* __restrict__ U, size_t su,
                                                 const double* __restrict__ P, size_t sp, double* __restrict__ A, size_t sa) {
  const long long pt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (pt >= d.npts) return;
  auto u = [&](int f) { return __ldg(U + (size_t)f * su + pt); };
  auto pr = [&](int f) { return __ldg(P + (size_t)f * sp + pt); };
  const double chi = u(CHI), ichi = 1.0 / chi;
  const double g[6] = {u(GXX) * ichi, u(GXY) * ichi, u(GXZ) * ichi, u(GYY) * ichi, u(GYZ) * ichi, u(GZZ) * ichi};   // gamma_ij
  const double isg = chi * sqrt(chi);                                                                              // 1 / sqrt(gamma)
  const double rho = pr(RHO), eps = pr(EPS), p = pr(PRESS), W = pr(WLOR);
  const double vu[3] = {pr(VX), pr(VY), pr(VZ)}, Bu[3] = {u(BXBAR) * isg, u(BYBAR) * isg, u(BZBAR) * isg};
  const double vl[3] = {g[0] * vu[0] + g[1] * vu[1] + g[2] * vu[2], g[1] * vu[0] + g[3] * vu[1] + g[4] * vu[2], g[2] * vu[0] + g[4] * vu[1] + g[5] * vu[2]};
  const double Bl[3] = {g[0] * Bu[0] + g[1] * Bu[1] + g[2] * Bu[2], g[1] * Bu[0] + g[3] * Bu[1] + g[4] * Bu[2], g[2] * Bu[0] + g[4] * Bu[1] + g[5] * Bu[2]};
  // E^i = -[ijk] v_j B_k / sqrt(gamma), E_i = gamma_ij E^j
  const double Eu[3] = {-(vl[1] * Bl[2] - vl[2] * Bl[1]) * isg, -(vl[2] * Bl[0] - vl[0] * Bl[2]) * isg, -(vl[0] * Bl[1] - vl[1] * Bl[0]) * isg};
  const double El[3] = {g[0] * Eu[0] + g[1] * Eu[1] + g[2] * Eu[2], g[1] * Eu[0] + g[3] * Eu[1] + g[4] * Eu[2], g[2] * Eu[0] + g[4] * Eu[1] + g[5] * Eu[2]};
  const double h = rho * (1.0 + eps) + p;
  double dpr, dpe, dpy = 0.0;
  if (TABLE) table_dp(par, rho, eps, pr(YE), dpr, dpe, dpy);
  else if (par.eos_kind == 0) { dpr = (par.eos_gamma - 1.0) * eps; dpe = (par.eos_gamma - 1.0) * rho; }
  else {                                                       // hybrid: p = K rho^G + (Gth - 1) rho (eps - a - K rho^(G-1) / (G-1)) in the piece of rho
    int i = 0;
    while (i < par.n_pieces - 1 && rho >= par.pp_rho[i]) ++i;
    const double G = par.pp_Gamma[i], x = par.pp_K[i] * pow(rho, G - 1.0), gth = par.eos_gamma_th - 1.0;   // x = p_cold / rho
    dpr = G * x + gth * (eps - par.pp_a[i] - x / (G - 1.0)) - gth * x;
    dpe = gth * rho;
  }
  double* a = A + pt;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    a[(A_BU + c) * sa] = Bu[c]; a[(A_VU + c) * sa] = vu[c]; a[(A_VL + c) * sa] = vl[c];
    a[(A_BL + c) * sa] = Bl[c]; a[(A_EL + c) * sa] = El[c]; a[(A_EU + c) * sa] = Eu[c];
  }
  a[A_VB * sa] = vl[0] * Bu[0] + vl[1] * Bu[1] + vl[2] * Bu[2];
  a[A_TH * sa] = h * W * W + (Bl[0] * Bu[0] + Bl[1] * Bu[1] + Bl[2] * Bu[2]);
  a[A_WM2 * sa] = 1.0 / (W * W);
  a[A_RHO * sa] = rho; a[A_EPS * sa] = eps; a[A_H * sa] = h; a[A_DPR * sa] = dpr; a[A_DPE * sa] = dpe;
  if (TABLE) { a[A_YE * sa] = pr(YE); a[A_DPY * sa] = dpy; }
  if (TABLE || FULL) a[A_D * sa] = rho * W;
  if (FULL) { a[A_CALE * sa] = h * W * W; a[A_DYE * sa] = rho * W * pr(YE); }
}

// The closed forms (A12)-(A16) from the point values a[] and the contracted gradient products, and the update of the work slot
struct LesDots { double dVB_B[3], dTH_v[3], dBv[3][3], sBv, sBBvB, sBvTh, sBB, sEE, svv, dWW, dWR, dWH, dPR_R, dPE_E, dRE, yterm; };   // yterm = grad(dp/dYe).grad Ye - (2/D) dp/dYe grad Ye.grad D

// the additional products of (A15) and (A17): grad B^k.grad B^i, grad v^k.grad v^i, grad E^k.grad E^i (symmetric, sym3 order) and grad D, grad(D Ye), grad calE . grad v^k
struct LesFull { double dBB[6], dvv[6], dEE[6], dD_v[3], dDY_v[3], dCE_v[3]; };

template <bool FULL>
__device__ __forceinline__ void les_closed_forms(const Dims& d, const Par& par, const double a[NAUX], const LesDots& D, const LesFull& X, const double gu[6],
                                                 double p, double chi, double al, const double* __restrict__ U, size_t su,
                                                 double* __restrict__ Wk, size_t sw, size_t pt, const double* wold = nullptr) {
  const double (&dVB_B)[3] = D.dVB_B; const double (&dTH_v)[3] = D.dTH_v; const double (&dBv)[3][3] = D.dBv;
  const double sBv = D.sBv, sBBvB = D.sBBvB, sBvTh = D.sBvTh, sBB = D.sBB, sEE = D.sEE, svv = D.svv;
  const double dWW = D.dWW, dWR = D.dWR, dWH = D.dWH, dPR_R = D.dPR_R, dPE_E = D.dPE_E, dRE = D.dRE;
  const double vB = a[A_VB], Th = a[A_TH], W2 = 1.0 / a[A_WM2], rho = a[A_RHO], h = a[A_H], dpr = a[A_DPR], dpe = a[A_DPE];
  const double calE = h * W2, iTh = 1.0 / Th, icalE = 1.0 / calE;
  const double E2 = a[A_EL] * a[A_EU] + a[A_EL + 1] * a[A_EU + 1] + a[A_EL + 2] * a[A_EU + 2];
  double Psi_v[3], vPsi = 0.0;
  const double brk = (Th * sBv + sBBvB - sBvTh) * icalE;
#pragma unroll
  for (int c = 0; c < 3; ++c) { Psi_v[c] = 2.0 * iTh * (dVB_B[c] - dTH_v[c] + a[A_BU + c] * brk); vPsi += a[A_VL + c] * Psi_v[c]; }
  // B_[i v_k] Psi_M^{ki} with Psi_M^{ki} = (4/Theta) [Theta gradB^[i.gradv^k] + B^[i gradB^k].grad(v.B) - B^[i gradv^k].gradTheta]
  double BvPsi = 0.0;
#pragma unroll
  for (int kk = 0; kk < 3; ++kk)
#pragma unroll
    for (int ii = 0; ii < 3; ++ii) {
      if (ii == kk) continue;
      const double psi = 2.0 * iTh * (Th * (dBv[ii][kk] - dBv[kk][ii]) + (a[A_BU + ii] * dVB_B[kk] - a[A_BU + kk] * dVB_B[ii])
                                      - (a[A_BU + ii] * dTH_v[kk] - a[A_BU + kk] * dTH_v[ii]));
      BvPsi += 0.5 * (a[A_BL + ii] * a[A_VL + kk] - a[A_BL + kk] * a[A_VL + ii]) * psi;
    }
  const double TmE = Th - E2;
  const double Psi_Th = Th / TmE * (sBB - sEE - BvPsi);
  const double Psi_A = W2 * (p * dpe + rho * rho * dpr);
  const double pref = calE * W2 * TmE / ((rho * calE - Psi_A) * TmE * W2 + Psi_A * Th);
  const double brace = rho * (dPR_R + dPE_E) - 2.0 * dpe * dRE
                       - (calE * dpe - Psi_A) * (0.25 * W2 * dWW + dWR / rho)
                       - 2.0 * a[A_WM2] * dpe * (sBB - W2 * W2 * dWH)
                       - (calE * dpe + Psi_A) * (vPsi + svv + W2 * dWW)
                       + Psi_Th * icalE * iTh * ((calE * dpe + Psi_A) * TmE - Psi_A * Th * a[A_WM2])
                       + rho * D.yterm;                     // the Y_e terms of (A12), inside the braces (reading R42); zero unless the EoS is tabulated
  const double H_Th = Psi_Th + Th / TmE * (pref * brace);                                   // (A13)
  double H_v[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) H_v[c] = Psi_v[c] - (a[A_VU + c] + vB * icalE * a[A_BU + c]) * H_Th * iTh;   // (A14)
  // (A11): xi = gamma^{1/3} Delta^2 / 24 = Delta^2 / (24 chi), sqrt(gamma) = chi^(-3/2)
  const double Delta2 = pow(d.dx * d.dy * d.dz, 2.0 / 3.0);
  const double sqrtg = 1.0 / (chi * sqrt(chi));
  const double fac0 = al * Delta2 / (24.0 * chi) * sqrtg, fac = fac0 * par.les_C_M;
  double HM[3][3];
#pragma unroll
  for (int kk = 0; kk < 3; ++kk)
#pragma unroll
    for (int ii = 0; ii < 3; ++ii) {
      HM[kk][ii] = 0.0;
      if (ii == kk) continue;
      HM[kk][ii] = (a[A_BU + ii] * H_v[kk] - a[A_BU + kk] * H_v[ii]) + 2.0 * (dBv[ii][kk] - dBv[kk][ii]);   // (A16)
      if (!FULL || par.les_C_M != 0.0) {
        double* w = Wk + (size_t)(11 * kk + 6 + ii) * sw + pt;
        *w = (wold ? wold[2 * kk + (ii > kk ? ii - 1 : ii)] : *w) + fac * HM[kk][ii];   // wold: the six fluxes fetched at kernel start (k_les_flux_tma)
      }
    }
  if constexpr (FULL) {
  // ---- (A15): H_N^k = 2 grad D . grad v^k + D H_v^k, the same with D Ye; fluxes of Dbar (field 0) and DYebar (field 1)
#pragma unroll
  for (int kk = 0; kk < 3; ++kk) {
    double* w = Wk + (size_t)(11 * kk) * sw + pt;
    if (par.les_C_N != 0.0) w[0] += fac0 * par.les_C_N * (2.0 * X.dD_v[kk] + a[A_D] * H_v[kk]);
    if (par.les_C_Y != 0.0) w[sw] += fac0 * par.les_C_Y * (2.0 * X.dDY_v[kk] + a[A_DYE] * H_v[kk]);
  }
  if (par.les_C_T == 0.0) return;
  // ---- (A17) with H_E_i = 1/2 sqrt(gamma) [ijk] H_M^{(dir k)(comp j)} (reading R45), the flux of Sbar_i is gamma_ij H_T^{kj}
  const double H_p = pref * brace;
  double HEl[3], HEu[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) { const int j = (c + 1) % 3, k = (c + 2) % 3; HEl[c] = 0.5 * sqrtg * (HM[k][j] - HM[j][k]); }
#pragma unroll
  for (int c = 0; c < 3; ++c) HEu[c] = gu[sym3(c, 0)] * HEl[0] + gu[sym3(c, 1)] * HEl[1] + gu[sym3(c, 2)] * HEl[2];
  const double EHE = a[A_EL] * HEu[0] + a[A_EL + 1] * HEu[1] + a[A_EL + 2] * HEu[2];
  const double trace = H_p + sBB + sEE + EHE;
  double HT[6];
#pragma unroll
  for (int kk = 0; kk < 3; ++kk)
#pragma unroll
    for (int ii = kk; ii < 3; ++ii) {
      const double vk = a[A_VU + kk], vi = a[A_VU + ii];
      const double first = vk * X.dCE_v[ii] + vi * X.dCE_v[kk] + calE * (0.5 * (vk * H_v[ii] + vi * H_v[kk]) + X.dvv[sym3(kk, ii)]) + vk * vi * H_p;
      const double second = X.dBB[sym3(kk, ii)] + X.dEE[sym3(kk, ii)] + 0.5 * (a[A_EU + kk] * HEu[ii] + a[A_EU + ii] * HEu[kk]);
      HT[sym3(kk, ii)] = 2.0 * first - 2.0 * second + (gu[sym3(kk, ii)] - vk * vi) * trace;
    }
  double gl[6];
  const double ichi = 1.0 / chi;
#pragma unroll
  for (int c = 0; c < 6; ++c) gl[c] = __ldg(U + (size_t)(GXX + c) * su + pt) * ichi;
#pragma unroll
  for (int kk = 0; kk < 3; ++kk)
#pragma unroll
    for (int ii = 0; ii < 3; ++ii) {
      double* w = Wk + (size_t)(11 * kk + 3 + ii) * sw + pt;
      *w += fac0 * par.les_C_T * (gl[sym3(ii, 0)] * HT[sym3(kk, 0)] + gl[sym3(ii, 1)] * HT[sym3(kk, 1)] + gl[sym3(ii, 2)] * HT[sym3(kk, 2)]);
    }
  }
}

template <bool FULL>
__global__ void __launch_bounds__(256, 1) k_les_flux(const __grid_constant__ Dims d, const __grid_constant__ Par par, const double* __restrict__ U, size_t su,
                                                  const double* __restrict__ P, size_t sp, const double* __restrict__ A, size_t sa,
                                                  double* __restrict__ Wk, size_t sw) {
  // a CTA owns a 16 x 4 x 4 block of points so that most y / z neighbours of a point are loaded by the same CTA and hit in L1
  const int i = 2 + blockIdx.x * 16 + threadIdx.x, j = 2 + blockIdx.y * 4 + threadIdx.y, k = 2 + blockIdx.z * 4 + threadIdx.z;
  if (i >= d.mx - 2 || j >= d.my - 2 || k >= d.mz - 2) return;
  const size_t pt = (size_t)k * d.sz + (size_t)j * d.sy + i;
  // inverse physical metric gamma^{mn} = chi gamma~^{mn}
  double gu[6];
  const double chi = __ldg(U + (size_t)CHI * su + pt), al = __ldg(U + (size_t)ALPHA * su + pt);
  {
    double g[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) g[c] = __ldg(U + (size_t)(GXX + c) * su + pt);
    const double s = chi / (g[0] * (g[3] * g[5] - g[4] * g[4]) - g[1] * (g[1] * g[5] - g[4] * g[2]) + g[2] * (g[1] * g[4] - g[3] * g[2]));
    gu[0] = (g[3] * g[5] - g[4] * g[4]) * s; gu[1] = (g[2] * g[4] - g[1] * g[5]) * s; gu[2] = (g[1] * g[4] - g[2] * g[3]) * s;
    gu[3] = (g[0] * g[5] - g[2] * g[2]) * s; gu[4] = (g[1] * g[2] - g[0] * g[4]) * s; gu[5] = (g[0] * g[3] - g[1] * g[1]) * s;
  }
  // Gradients are streamed field by field (Eq. 60) and contracted at once: only the raised gradients gamma^{mn} d_n f of a few anchor
  // fields (B^c, Theta, then W^-2, rho, eps) stay in registers, so that grad f . grad g = sum_m d_m f (gamma^{mn} d_n g) costs three FMAs and the
  // kernel holds ~60 doubles instead of the 180 that all 26 gradients in both index positions would take.
  const double c12[3] = {1.0 / (12.0 * d.dx), 1.0 / (12.0 * d.dy), 1.0 / (12.0 * d.dz)};
  const long long st[3] = {1, d.sy, d.sz};
  auto val = [&](int f) { return __ldg(A + (size_t)f * sa + pt); };
  auto grad = [&](int f, double g[3]) {
    const double* s = A + (size_t)f * sa + pt;
#pragma unroll
    for (int m = 0; m < 3; ++m) g[m] = (8.0 * (__ldg(s + st[m]) - __ldg(s - st[m])) - (__ldg(s + 2 * st[m]) - __ldg(s - 2 * st[m]))) * c12[m];
  };
  auto raise = [&](const double g[3], double r[3]) {
    r[0] = gu[0] * g[0] + gu[1] * g[1] + gu[2] * g[2];
    r[1] = gu[1] * g[0] + gu[3] * g[1] + gu[4] * g[2];
    r[2] = gu[2] * g[0] + gu[4] * g[1] + gu[5] * g[2];
  };
  auto dotp = [](const double g[3], const double r[3]) { return g[0] * r[0] + g[1] * r[1] + g[2] * r[2]; };
  double a[NAUX];                               // point values the closed forms use (vector components; the scalars are fetched where needed)
#pragma unroll
  for (int f = 0; f < A_VB; ++f) a[f] = val(f);
  double uB[3][3], uTH[3], t[3], t2[3], r[3];
  LesFull X;
  double uVa[FULL ? 3 : 1][3], uEa[FULL ? 3 : 1][3];   // FULL: the raised gradients of every v^c and E^c stay for grad v^k.grad v^i, grad E^k.grad E^i
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    grad(A_BU + c, t); raise(t, uB[c]);
    if (FULL)
#pragma unroll
      for (int e = 0; e <= c; ++e) X.dBB[sym3(e, c)] = dotp(t, uB[e]);
  }
  grad(A_TH, t); raise(t, uTH);
  double dVB_B[3], dTH_v[3], dBv[3][3];         // grad(v.B).grad B^k, grad Theta.grad v^k, grad B^i.grad v^k
  grad(A_VB, t);
#pragma unroll
  for (int c = 0; c < 3; ++c) dVB_B[c] = dotp(t, uB[c]);
  double sBv = 0.0, sBBvB = 0.0, sBvTh = 0.0, sBB = 0.0, sEE = 0.0, svv = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    grad(A_VU + c, t);
    dTH_v[c] = dotp(t, uTH);
#pragma unroll
    for (int e = 0; e < 3; ++e) dBv[e][c] = dotp(t, uB[e]);
    raise(t, r);
    if (FULL) {
#pragma unroll
      for (int m = 0; m < 3; ++m) uVa[FULL ? c : 0][m] = r[m];
#pragma unroll
      for (int e = 0; e <= c; ++e) X.dvv[sym3(e, c)] = dotp(t, uVa[FULL ? e : 0]);
    }
    grad(A_VL + c, t2);
    svv += dotp(t2, r);
    sBv += dotp(t2, uB[c]);
    sBvTh += a[A_BU + c] * dotp(t2, uTH);
    grad(A_BL + c, t);
    sBB += dotp(t, uB[c]);
    grad(A_EU + c, t); raise(t, r);
    if (FULL) {
#pragma unroll
      for (int m = 0; m < 3; ++m) uEa[FULL ? c : 0][m] = r[m];
#pragma unroll
      for (int e = 0; e <= c; ++e) X.dEE[sym3(e, c)] = dotp(t, uEa[FULL ? e : 0]);
    }
    grad(A_EL + c, t2);
    sEE += dotp(t2, r);
    sBBvB += a[A_BL + c] * dVB_B[c];
  }
  double dWW, dWR, dWH, dPR_R, dPE_E, dRE;
  {
    double uW[3], uR[3], uE[3];
    grad(A_WM2, t); raise(t, uW); dWW = dotp(t, uW);
    grad(A_RHO, t); dWR = dotp(t, uW); raise(t, uR);
    grad(A_H, t); dWH = dotp(t, uW);
    grad(A_DPR, t); dPR_R = dotp(t, uR);
    grad(A_EPS, t); dRE = dotp(t, uR); raise(t, uE);
    grad(A_DPE, t); dPE_E = dotp(t, uE);
  }
  const double p = __ldg(P + (size_t)PRESS * sp + pt);
  a[A_VB] = val(A_VB); a[A_TH] = val(A_TH); a[A_WM2] = val(A_WM2); a[A_RHO] = val(A_RHO); a[A_H] = val(A_H); a[A_DPR] = val(A_DPR); a[A_DPE] = val(A_DPE);
  LesDots D;
#pragma unroll
  for (int c = 0; c < 3; ++c) { D.dVB_B[c] = dVB_B[c]; D.dTH_v[c] = dTH_v[c]; for (int e = 0; e < 3; ++e) D.dBv[c][e] = dBv[c][e]; }
  D.sBv = sBv; D.sBBvB = sBBvB; D.sBvTh = sBvTh; D.sBB = sBB; D.sEE = sEE; D.svv = svv;
  D.dWW = dWW; D.dWR = dWR; D.dWH = dWH; D.dPR_R = dPR_R; D.dPE_E = dPE_E; D.dRE = dRE;
  D.yterm = 0.0;
  if (par.eos_kind == 2) {
    double uY[3];
    grad(A_YE, t); raise(t, uY);
    grad(A_DPY, t2); const double dPY_Y = dotp(t2, uY);
    grad(A_D, t2);
    D.yterm = dPY_Y - 2.0 / val(A_D) * val(A_DPY) * dotp(t2, uY);
  }
  if (FULL) {
    a[A_D] = val(A_D); a[A_DYE] = val(A_DYE);
    grad(A_D, t);
#pragma unroll
    for (int c = 0; c < 3; ++c) X.dD_v[c] = dotp(t, uVa[FULL ? c : 0]);
    grad(A_DYE, t);
#pragma unroll
    for (int c = 0; c < 3; ++c) X.dDY_v[c] = dotp(t, uVa[FULL ? c : 0]);
    grad(A_CALE, t);
#pragma unroll
    for (int c = 0; c < 3; ++c) X.dCE_v[c] = dotp(t, uVa[FULL ? c : 0]);
  }
  les_closed_forms<FULL>(d, par, a, D, X, gu, p, chi, al, U, su, Wk, sw, pt);
}


// ---------------------------------------------------------------------------------------------------------------
// The same computation with the auxiliary fields staged by the copy engine (default whenever the LESWORK slot admits a tensor map):
// a CTA of 256 threads owns a 16 x 4 x 4 block of points; the 26 fields pass one at a time, in the order the streaming contraction
// needs them, in 5 groups of 5-6 fields through three shared-memory buffers of 20 x 8 x 8 tiles (block + halo 2; the copies run two groups ahead) filled by
// cp.async.bulk.tensor with mbarrier completion, so the 12 stencil operands of a field are shared-memory loads with compile-time
// offsets and the copy of group g+1 overlaps the arithmetic on group g (one barrier per group: a barrier per field leaves too little work
// between barriers, measured 32.6 vs 29.2 ms per step for the L1 version at c1_256). (k_les_flux above fetches them through L1/L2 with one exposed latency per field at 8 warps/SM.)
// ---------------------------------------------------------------------------------------------------------------
constexpr int LX = 16, LY = 4, LZ = 4, LH = 2, LSX = LX + 2 * LH, LSY = LY + 2 * LH, LSZ = LZ + 2 * LH, LTILE = LSX * LSY * LSZ, LGMAX = 6, LNBUF = 3;
// the fields pass in 5 groups (one barrier and one mbarrier wait per group, not per field): {B^c, Theta, v.B}, three times {v^c, v_c, B_c, E^c, E_c}, the 6 scalars
// then, in the order of LORDER: {Ye, dp/dYe, D} with the tabulated EoS only, {calE, D Ye} with FULL only (without the table: one group {D, calE, D Ye})
template <int... Is, class F> __device__ __forceinline__ void static_for(std::integer_sequence<int, Is...>, F&& f) { (f(std::integral_constant<int, Is>{}), ...); }
template <bool TABLE, bool FULL> struct LGroups {
  static constexpr int N = 5 + (TABLE ? 1 : 0) + (FULL ? 1 : 0);
  __host__ __device__ static constexpr int start(int g) { return g < 5 ? 5 * g : g == 5 ? (TABLE ? 26 : 28) : 29; }
  __host__ __device__ static constexpr int end(int g) { return g < 4 ? 5 * (g + 1) : g == 4 ? 26 : g == 5 ? (TABLE ? 29 : 31) : 31; }
};
constexpr size_t LES_SMEM = (size_t)LNBUF * LGMAX * LTILE * sizeof(double) + 64;   // three buffers: the copies run two groups ahead of the arithmetic
// order of passage: anchors B^c, Theta; v.B; then per component c: v^c, v_c, B_c, E^c, E_c; then W^-2, rho, h, dp/drho, eps, dp/deps
__device__ constexpr int LORDER[NAUX] = {A_BU, A_BU + 1, A_BU + 2, A_TH, A_VB,
                                         A_VU, A_VL, A_BL, A_EU, A_EL, A_VU + 1, A_VL + 1, A_BL + 1, A_EU + 1, A_EL + 1, A_VU + 2, A_VL + 2, A_BL + 2, A_EU + 2, A_EL + 2,
                                         A_WM2, A_RHO, A_H, A_DPR, A_EPS, A_DPE, A_YE, A_DPY, A_D, A_CALE, A_DYE};

template <bool TABLE, bool FULL>
__global__ void __launch_bounds__(LX * LY * LZ, 1) k_les_flux_tma(const __grid_constant__ Dims d, const __grid_constant__ Par par, const double* __restrict__ U, size_t su,
                                                                  const double* __restrict__ P, size_t sp, double* __restrict__ Wk, size_t sw,
                                                                  const __grid_constant__ CUtensorMap tmap) {
  static_assert((LTILE * sizeof(double)) % 128 == 0, "TMA destination tiles must stay 128-byte aligned");
  using LG = LGroups<TABLE, FULL>;
  extern __shared__ __align__(128) double ring[];
  uint64_t* full = (uint64_t*)(ring + LNBUF * LGMAX * LTILE);
  const int tid = threadIdx.x, tx = tid % LX, ty = (tid / LX) % LY, tz = tid / (LX * LY);
  const int i0 = 2 + blockIdx.x * LX, j0 = 2 + blockIdx.y * LY, k0 = 2 + blockIdx.z * LZ;      // array indices of the block's first point
  const int i = i0 + tx, j = j0 + ty, k = k0 + tz;
  const bool inside = i < d.mx - 2 && j < d.my - 2 && k < d.mz - 2;
  const size_t pt = (size_t)min(k, d.mz - 3) * d.sz + (size_t)min(j, d.my - 3) * d.sy + min(i, d.mx - 3);
  if (tid == 0) {
#pragma unroll
    for (int b = 0; b < LNBUF; ++b) mbar_init(full + b, 1);
    mbar_fence_init();
  }
  __syncthreads();
  auto issue = [&](int g) {                       // the box origin i0 - 2 = 16 blockIdx.x is even: on a 16-byte boundary
    if (tid == 0) {
      const int n0 = LG::start(g), n1 = LG::end(g);
      mbar_expect_tx(full + g % LNBUF, (unsigned)(n1 - n0) * LTILE * (unsigned)sizeof(double));
      for (int n = n0; n < n1; ++n) tma_load_4d(ring + ((g % LNBUF) * LGMAX + (n - n0)) * LTILE, &tmap, full + g % LNBUF, i0 - LH, j0 - LH, k0 - LH, LORDER[n]);
    }
  };
  issue(0);
  issue(1);
  // the fluxes this thread adds its SGS terms to at the very end (read-modify-write of the work slot) are pulled into L1 now: with one CTA per SM nothing
  // else would cover that HBM round trip (it was 40 % of the kernel's stall samples)
  double wold[6];                                  // C_M only: the six fluxes of Bbar^i (direction k != i) are fetched into registers right away
  if (!FULL) {
#pragma unroll
    for (int kk = 0; kk < 3; ++kk)
#pragma unroll
      for (int ii = 0; ii < 3; ++ii)
        if (ii != kk) wold[2 * kk + (ii > kk ? ii - 1 : ii)] = Wk[(size_t)(11 * kk + 6 + ii) * sw + pt];
  } else if (inside) {                             // FULL (no registers left): Dbar, DYebar, Sbar_i, Bbar^i fluxes (not taubar) as L1 prefetches
    auto pf = [](const double* a) { asm volatile("prefetch.global.L1 [%0];" ::"l"(a)); };
#pragma unroll
    for (int kk = 0; kk < 3; ++kk)
#pragma unroll
      for (int f = 0; f < 9; ++f) {
        if (f == 2 || f == 6 + kk) continue;
        pf(Wk + (size_t)(11 * kk + f) * sw + pt);
      }
  }
  double gu[6];
  const double chi = __ldg(U + (size_t)CHI * su + pt), al = __ldg(U + (size_t)ALPHA * su + pt);
  // the point values of the metric are requested here and first used after the first group of fields has passed (its gradients are kept lower-index until
  // then): with one CTA per SM nothing else would cover this HBM round trip
  double gm[6];
#pragma unroll
  for (int c = 0; c < 6; ++c) gm[c] = __ldg(U + (size_t)(GXX + c) * su + pt);
  auto inverse_metric = [&]() {
    const double s = chi / (gm[0] * (gm[3] * gm[5] - gm[4] * gm[4]) - gm[1] * (gm[1] * gm[5] - gm[4] * gm[2]) + gm[2] * (gm[1] * gm[4] - gm[3] * gm[2]));
    gu[0] = (gm[3] * gm[5] - gm[4] * gm[4]) * s; gu[1] = (gm[2] * gm[4] - gm[1] * gm[5]) * s; gu[2] = (gm[1] * gm[4] - gm[2] * gm[3]) * s;
    gu[3] = (gm[0] * gm[5] - gm[2] * gm[2]) * s; gu[4] = (gm[1] * gm[2] - gm[0] * gm[4]) * s; gu[5] = (gm[0] * gm[3] - gm[1] * gm[1]) * s;
  };
  const double p = __ldg(P + (size_t)PRESS * sp + pt);
  const double c12[3] = {1.0 / (12.0 * d.dx), 1.0 / (12.0 * d.dy), 1.0 / (12.0 * d.dz)};
  auto raise = [&](const double g[3], double r[3]) {
    r[0] = gu[0] * g[0] + gu[1] * g[1] + gu[2] * g[2];
    r[1] = gu[1] * g[0] + gu[3] * g[1] + gu[4] * g[2];
    r[2] = gu[2] * g[0] + gu[4] * g[1] + gu[5] * g[2];
  };
  auto dotp = [](const double g[3], const double r[3]) { return g[0] * r[0] + g[1] * r[1] + g[2] * r[2]; };
  const int ctr = ((tz + LH) * LSY + (ty + LH)) * LSX + (tx + LH);
  double a[NAUX];
  LesDots D;
  D.sBv = D.sBBvB = D.sBvTh = D.sBB = D.sEE = D.svv = 0.0;
  D.yterm = 0.0;
  LesFull X;
  // raised gradients of the anchors: B^c, Theta, v^c and E^c (FULL: every component stays, for (A17)), the current W^-2 / eps / Ye, rho
  double uB[3][3], uTH[3], gVB[3], uV[FULL ? 3 : 1][3], uE[FULL ? 3 : 1][3], uX[3], uR[3];
  // the groups are expanded at compile time (a fold over their indices: `#pragma unroll` gives up on the seven groups of <TABLE, FULL> and leaves a[], D, X in local memory)
  auto group = [&](auto G) {
    constexpr int g5 = decltype(G)::value;
    __syncthreads();                                 // everybody is done reading the buffer the next copy overwrites
    if (g5 + 2 < LG::N) issue(g5 + 2);             // into the buffer group g5 - 1 has just released
    mbar_wait(full + g5 % LNBUF, (g5 / LNBUF) & 1);
#pragma unroll
   for (int n = LG::start(g5); n < LG::end(g5); ++n) {
    const double* s = ring + ((g5 % LNBUF) * LGMAX + (n - LG::start(g5))) * LTILE + ctr;
    constexpr int OX = 1, OY = LSX, OZ = LSX * LSY;
    const int f = LORDER[n];
    a[f] = s[0];
    double g[3];
    g[0] = (8.0 * (s[OX] - s[-OX]) - (s[2 * OX] - s[-2 * OX])) * c12[0];
    g[1] = (8.0 * (s[OY] - s[-OY]) - (s[2 * OY] - s[-2 * OY])) * c12[1];
    g[2] = (8.0 * (s[OZ] - s[-OZ]) - (s[2 * OZ] - s[-2 * OZ])) * c12[2];
    if (n == 5) {                                                          // first field after the anchors: now the inverse metric is needed
      inverse_metric();
#pragma unroll
      for (int c = 0; c < 3; ++c) {                                        // raise grad B^c in place (FULL: grad B^e . grad B^c on the way)
        const double lo[3] = {uB[c][0], uB[c][1], uB[c][2]};
        raise(lo, uB[c]);
        if (FULL)
#pragma unroll
          for (int e = 0; e <= c; ++e) X.dBB[sym3(e, c)] = dotp(lo, uB[e]);
        D.dVB_B[c] = dotp(gVB, uB[c]);
      }
      const double lo[3] = {uTH[0], uTH[1], uTH[2]};
      raise(lo, uTH);
    }
    if (n < 3) { uB[n][0] = g[0]; uB[n][1] = g[1]; uB[n][2] = g[2]; }      // B^c: kept lower-index until n == 5
    else if (n == 3) { uTH[0] = g[0]; uTH[1] = g[1]; uTH[2] = g[2]; }      // Theta
    else if (n == 4) { gVB[0] = g[0]; gVB[1] = g[1]; gVB[2] = g[2]; }      // v.B
    else if (n < 20) {
      const int c = (n - 5) / 5, w = (n - 5) % 5;
      if (w == 0) {                                                        // v^c
        D.dTH_v[c] = dotp(g, uTH);
#pragma unroll
        for (int e = 0; e < 3; ++e) D.dBv[e][c] = dotp(g, uB[e]);
        raise(g, uV[FULL ? c : 0]);
        if (FULL)
#pragma unroll
          for (int e = 0; e <= c; ++e) X.dvv[sym3(e, c)] = dotp(g, uV[FULL ? e : 0]);
      } else if (w == 1) {                                                 // v_c
        D.svv += dotp(g, uV[FULL ? c : 0]);
        D.sBv += dotp(g, uB[c]);
        D.sBvTh += a[A_BU + c] * dotp(g, uTH);
      } else if (w == 2) {                                                 // B_c
        D.sBB += dotp(g, uB[c]);
        D.sBBvB += a[A_BL + c] * D.dVB_B[c];
      } else if (w == 3) {                                                 // E^c
        raise(g, uE[FULL ? c : 0]);
        if (FULL)
#pragma unroll
          for (int e = 0; e <= c; ++e) X.dEE[sym3(e, c)] = dotp(g, uE[FULL ? e : 0]);
      } else D.sEE += dotp(g, uE[FULL ? c : 0]);                           // E_c
    } else if (n == 20) { raise(g, uX); D.dWW = dotp(g, uX); }             // W^-2
    else if (n == 21) { D.dWR = dotp(g, uX); raise(g, uR); }               // rho
    else if (n == 22) D.dWH = dotp(g, uX);                                 // h
    else if (n == 23) D.dPR_R = dotp(g, uR);                               // dp/drho
    else if (n == 24) { D.dRE = dotp(g, uR); raise(g, uX); }               // eps
    else if (n == 25) D.dPE_E = dotp(g, uX);                               // dp/deps
    else if (n == 26) raise(g, uX);                                        // Ye
    else if (n == 27) D.yterm = dotp(g, uX);                               // dp/dYe
    else if (n == 28) {                                                    // D
      if (TABLE) D.yterm -= 2.0 / a[A_D] * a[A_DPY] * dotp(g, uX);
      if (FULL)
#pragma unroll
        for (int c = 0; c < 3; ++c) X.dD_v[c] = dotp(g, uV[FULL ? c : 0]);
    } else if (n == 29) {                                                  // calE
#pragma unroll
      for (int c = 0; c < 3; ++c) X.dCE_v[c] = dotp(g, uV[FULL ? c : 0]);
    } else {                                                               // D Ye
#pragma unroll
      for (int c = 0; c < 3; ++c) X.dDY_v[c] = dotp(g, uV[FULL ? c : 0]);
    }
   }
  };
  static_for(std::make_integer_sequence<int, LG::N>{}, group);
  if (inside) les_closed_forms<FULL>(d, par, a, D, X, gu, p, chi, al, U, su, Wk, sw, pt, FULL ? nullptr : wold);
}

}  // namespace

template <bool TABLE, bool FULL>
static cudaError_t launch_les_t(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* A, size_t sa,
                                double* Wk, size_t sw, cudaStream_t s) {
  k_les_aux<TABLE, FULL><<<(unsigned)((d.npts + 127) / 128), 128, 0, s>>>(d, par, U, su, P, sp, A, sa);
  if (d.mx > 4 && d.my > 4 && d.mz > 4) {
    dim3 grid((d.mx - 4 + 15) / 16, (d.my - 4 + 3) / 4, (d.mz - 4 + 3) / 4), block(16, 4, 4);
    CUtensorMap map;
    static int attr[64] = {};                                  // one per instantiation
    int dev = 0;
    cudaGetDevice(&dev);
    bool tma = dev >= 0 && dev < 64 && make_tensor_map_4d(d, A, sa, FULL ? NAUX : TABLE ? A_D + 1 : NAUX_NOYE, LSX, LSY, LSZ, &map);
    if (tma && !attr[dev]) {
      tma = cudaFuncSetAttribute(k_les_flux_tma<TABLE, FULL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LES_SMEM) == cudaSuccess;
      attr[dev] = tma;
    }
    if (tma) k_les_flux_tma<TABLE, FULL><<<grid, LX * LY * LZ, LES_SMEM, s>>>(d, par, U, su, P, sp, Wk, sw, map);
    else k_les_flux<FULL><<<grid, block, 0, s>>>(d, par, U, su, P, sp, A, sa, Wk, sw);
  }
  return cudaGetLastError();
}

cudaError_t launch_les(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* A, size_t sa,
                       double* Wk, size_t sw, cudaStream_t s) {
  const bool full = par.les_C_N != 0.0 || par.les_C_Y != 0.0 || par.les_C_T != 0.0, table = par.eos_kind == 2;
  if (table) return full ? launch_les_t<true, true>(d, par, U, su, P, sp, A, sa, Wk, sw, s) : launch_les_t<true, false>(d, par, U, su, P, sp, A, sa, Wk, sw, s);
  return full ? launch_les_t<false, true>(d, par, U, su, P, sp, A, sa, Wk, sw, s) : launch_les_t<false, false>(d, par, U, su, P, sp, A, sa, Wk, sw, s);
}

}  // namespace mhd
