// LES gradient sub-grid-scale tensor of the induction equation: PAPER.md Sec. II B l.252-256 and App. A,
// Eqs. (A11)-(A17) l.855-882, coefficient C_M (the paper's production setting: C_M = 8, the other coefficients 0, l.863).
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
// EoS derivatives: analytic for the ideal gas and the hybrid piecewise polytrope (l.882); the tabulated EoS is not supported here.
#include "mhd_internal.cuh"

namespace mhd {

namespace {

enum { A_BU = 0, A_VU = 3, A_VL = 6, A_BL = 9, A_EL = 12, A_EU = 15, A_VB = 18, A_TH = 19, A_WM2 = 20, A_RHO = 21, A_EPS = 22, A_H = 23,
       A_DPR = 24, A_DPE = 25, NAUX = MHD_NLESWORK };

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
  double dpr, dpe;
  if (par.eos_kind == 0) { dpr = (par.eos_gamma - 1.0) * eps; dpe = (par.eos_gamma - 1.0) * rho; }
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
}

__global__ void __launch_bounds__(128) k_les_flux(const __grid_constant__ Dims d, const __grid_constant__ Par par, const double* __restrict__ U, size_t su,
                                                  const double* __restrict__ P, size_t sp, const double* __restrict__ A, size_t sa,
                                                  double* __restrict__ Wk, size_t sw) {
  const int i = 2 + blockIdx.x * blockDim.x + threadIdx.x, j = 2 + blockIdx.y, k = 2 + blockIdx.z;
  if (i >= d.mx - 2) return;
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
  // point values and gradients: dl = d_m f (Eq. 60), du = gamma^{mn} d_n f, so that grad f . grad g = sum_m dl_f[m] du_g[m]
  double a[NAUX], dl[NAUX][3], du[NAUX][3];
  const double c12[3] = {1.0 / (12.0 * d.dx), 1.0 / (12.0 * d.dy), 1.0 / (12.0 * d.dz)};
  const long long st[3] = {1, d.sy, d.sz};
#pragma unroll
  for (int f = 0; f < NAUX; ++f) {
    const double* s = A + (size_t)f * sa + pt;
    a[f] = __ldg(s);
#pragma unroll
    for (int m = 0; m < 3; ++m) dl[f][m] = (8.0 * (__ldg(s + st[m]) - __ldg(s - st[m])) - (__ldg(s + 2 * st[m]) - __ldg(s - 2 * st[m]))) * c12[m];
    du[f][0] = gu[0] * dl[f][0] + gu[1] * dl[f][1] + gu[2] * dl[f][2];
    du[f][1] = gu[1] * dl[f][0] + gu[3] * dl[f][1] + gu[4] * dl[f][2];
    du[f][2] = gu[2] * dl[f][0] + gu[4] * dl[f][1] + gu[5] * dl[f][2];
  }
  auto dot = [&](int f, int g) { return dl[f][0] * du[g][0] + dl[f][1] * du[g][1] + dl[f][2] * du[g][2]; };
  const double p = __ldg(P + (size_t)PRESS * sp + pt);
  const double vB = a[A_VB], Th = a[A_TH], W2 = 1.0 / a[A_WM2], rho = a[A_RHO], h = a[A_H], dpr = a[A_DPR], dpe = a[A_DPE];
  const double calE = h * W2, iTh = 1.0 / Th, icalE = 1.0 / calE;
  const double E2 = a[A_EL] * a[A_EU] + a[A_EL + 1] * a[A_EU + 1] + a[A_EL + 2] * a[A_EU + 2];
  // products shared between (A12)-(A16)
  double dVB_B[3], dTH_v[3], dBv[3][3];        // grad(v.B).grad B^k, grad Theta.grad v^k, grad B^i.grad v^k
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    dVB_B[c] = dot(A_VB, A_BU + c);
    dTH_v[c] = dot(A_TH, A_VU + c);
#pragma unroll
    for (int e = 0; e < 3; ++e) dBv[c][e] = dot(A_BU + c, A_VU + e);
  }
  double sBv = 0.0, sBBvB = 0.0, sBvTh = 0.0, sBB = 0.0, sEE = 0.0, svv = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    sBv += dot(A_BU + c, A_VL + c);
    sBBvB += a[A_BL + c] * dVB_B[c];
    sBvTh += a[A_BU + c] * dot(A_VL + c, A_TH);
    sBB += dot(A_BL + c, A_BU + c);
    sEE += dot(A_EL + c, A_EU + c);
    svv += dot(A_VL + c, A_VU + c);
  }
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
  const double dWW = dot(A_WM2, A_WM2);
  const double pref = calE * W2 * TmE / ((rho * calE - Psi_A) * TmE * W2 + Psi_A * Th);
  const double brace = rho * (dot(A_DPR, A_RHO) + dot(A_DPE, A_EPS)) - 2.0 * dpe * dot(A_RHO, A_EPS)
                       - (calE * dpe - Psi_A) * (0.25 * W2 * dWW + dot(A_WM2, A_RHO) / rho)
                       - 2.0 * a[A_WM2] * dpe * (sBB - W2 * W2 * dot(A_WM2, A_H))
                       - (calE * dpe + Psi_A) * (vPsi + svv + W2 * dWW)
                       + Psi_Th * icalE * iTh * ((calE * dpe + Psi_A) * TmE - Psi_A * Th * a[A_WM2]);
  const double H_Th = Psi_Th + Th / TmE * (pref * brace);                                   // (A13)
  double H_v[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) H_v[c] = Psi_v[c] - (a[A_VU + c] + vB * icalE * a[A_BU + c]) * H_Th * iTh;   // (A14)
  // (A11): xi = gamma^{1/3} Delta^2 / 24 = Delta^2 / (24 chi), sqrt(gamma) = chi^(-3/2)
  const double Delta2 = pow(d.dx * d.dy * d.dz, 2.0 / 3.0);
  const double fac = al * par.les_C_M * Delta2 / (24.0 * chi) / (chi * sqrt(chi));
#pragma unroll
  for (int kk = 0; kk < 3; ++kk)
#pragma unroll
    for (int ii = 0; ii < 3; ++ii) {
      if (ii == kk) continue;
      const double HM = (a[A_BU + ii] * H_v[kk] - a[A_BU + kk] * H_v[ii]) + 2.0 * (dBv[ii][kk] - dBv[kk][ii]);   // (A16)
      double* w = Wk + (size_t)(11 * kk + 6 + ii) * sw + pt;
      *w += fac * HM;
    }
}

}  // namespace

cudaError_t launch_les(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* A, size_t sa,
                       double* Wk, size_t sw, cudaStream_t s) {
  k_les_aux<<<(unsigned)((d.npts + 127) / 128), 128, 0, s>>>(d, par, U, su, P, sp, A, sa);
  if (d.mx > 4 && d.my > 4 && d.mz > 4) {
    dim3 grid((d.mx - 4 + 127) / 128, d.my - 4, d.mz - 4);
    k_les_flux<<<grid, 128, 0, s>>>(d, par, U, su, P, sp, A, sa, Wk, sw);
  }
  return cudaGetLastError();
}

}  // namespace mhd
