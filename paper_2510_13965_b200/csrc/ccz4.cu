// a3-a5 (+ a4, a8): CCZ4 + gauge right-hand side, Eqs. (13)-(26) l.141-202, with the 4th-order centred
// differences of Eqs. (60)-(62), the one-sided advective stencils (l.454-456), Kreiss-Oliger dissipation (l.460),
// the matter projections tau, S_i, S_ij (l.188-192, l.260) and — because they need the very same derivatives of
// alpha, beta^i, gamma~_ij, chi — the geometric and divergence-cleaning SOURCES of the GRMHD system (right-hand
// sides of Eq. 32, l.256). Output: K_f for the 22 spacetime fields, and the source part of the 10 fluid fields
// (the flux kernels of flux.cu subtract the flux divergence afterwards).
//
// One thread per interior point, x-contiguous warps. All stencils are evaluated on differences (note N1 of
// DESIGN.md): algebraically identical to the printed coefficients, exact zeros in flat space, no cancellation noise.
// The algebra is staged (Christoffels -> Ricci -> lapse Hessian -> shift terms -> curvature terms -> outputs) so
// that second derivatives are contracted as soon as they are formed and never all live at once.
#include "mhd_internal.cuh"

namespace mhd {

namespace {

__device__ __forceinline__ int sym(int i, int j) { return i <= j ? (i * (5 - i)) / 2 + j : (j * (5 - j)) / 2 + i; }   // (0,0)=0 (0,1)=1 (0,2)=2 (1,1)=3 (1,2)=4 (2,2)=5

struct Stencil {
  long long s[3];      // strides
  double i12h[3];      // 1/(12 h)
  double i12h2[3];     // 1/(12 h^2)
  double i64h[3];      // 1/(64 h)
};

__device__ __forceinline__ double ld(const double* p) { return __ldg(p); }

// Eq. (60)
__device__ __forceinline__ double D1(const double* u, long long s, double i12h) {
  return (8.0 * (ld(u + s) - ld(u - s)) - (ld(u + 2 * s) - ld(u - 2 * s))) * i12h;
}
// Eq. (62)
__device__ __forceinline__ double D2(const double* u, long long s, double i12h2) {
  const double u0 = ld(u);
  return (16.0 * ((ld(u + s) - u0) + (ld(u - s) - u0)) - ((ld(u + 2 * s) - u0) + (ld(u - 2 * s) - u0))) * i12h2;
}
// Eq. (61): D_b (D_a u)
__device__ __forceinline__ double D11(const double* u, long long sa, double ia, long long sb, double ib) {
  const double p1 = D1(u + sb, sa, ia), m1 = D1(u - sb, sa, ia), p2 = D1(u + 2 * sb, sa, ia), m2 = D1(u - 2 * sb, sa, ia);
  return (8.0 * (p1 - m1) - (p2 - m2)) * ib;
}
// beta^k D_k u with the one-sided stencils of l.454-456 (beta >= 0 takes the "beta > 0" branch) + KO of l.460, all 3 axes
__device__ __forceinline__ double adv_ko(const double* u, const Stencil& st, const double be[3], double sigma) {
  const double u0 = ld(u);
  double acc = 0.0;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const long long s = st.s[k];
    const double m3 = ld(u - 3 * s) - u0, m2 = ld(u - 2 * s) - u0, m1 = ld(u - s) - u0;
    const double p1 = ld(u + s) - u0, p2 = ld(u + 2 * s) - u0, p3 = ld(u + 3 * s) - u0;
    const double up = (p3 - 6.0 * p2 + 18.0 * p1 - 3.0 * m1);       // beta > 0
    const double dn = (-m3 + 6.0 * m2 - 18.0 * m1 + 3.0 * p1);      // beta < 0
    acc += be[k] * ((be[k] < 0.0 ? dn : up) * st.i12h[k]);
    acc += sigma * st.i64h[k] * ((m3 + p3) - 6.0 * (m2 + p2) + 15.0 * (m1 + p1));
  }
  return acc;
}

}  // namespace

__global__ void __launch_bounds__(256, 1)
k_rhs_ccz4(const __grid_constant__ Dims d, const __grid_constant__ Par par, const double* __restrict__ U, size_t su,
           const double* __restrict__ P, size_t sp, double* __restrict__ K, size_t sk) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i >= d.nx || j >= d.ny || k >= d.nz) return;
  const size_t pt = (size_t)(k + d.ng) * d.sz + (size_t)(j + d.ng) * d.sy + (i + d.ng);
  Stencil st;
  st.s[0] = 1; st.s[1] = d.sy; st.s[2] = d.sz;
  {
    const double h[3] = {d.dx, d.dy, d.dz};
#pragma unroll
    for (int a = 0; a < 3; ++a) { st.i12h[a] = 1.0 / (12.0 * h[a]); st.i12h2[a] = 1.0 / (12.0 * h[a] * h[a]); st.i64h[a] = 1.0 / (64.0 * h[a]); }
  }
  auto F = [&](int f) { return U + (size_t)f * su + pt; };
  auto d1 = [&](int f, int a) { return D1(F(f), st.s[a], st.i12h[a]); };
  auto d2 = [&](int f, int a, int b) {
    return a == b ? D2(F(f), st.s[a], st.i12h2[a]) : D11(F(f), st.s[a], st.i12h[a], st.s[b], st.i12h[b]);
  };
  auto OUT = [&](int f) -> double& { return K[(size_t)f * sk + pt]; };

  // ---- point values
  double g[6], gi[6];
#pragma unroll
  for (int a = 0; a < 6; ++a) g[a] = ld(F(GXX + a));
  const double chi = ld(F(CHI)), al = ld(F(ALPHA));
  const double be[3] = {ld(F(BETAX)), ld(F(BETAY)), ld(F(BETAZ))};
  const double detg = g[0] * (g[3] * g[5] - g[4] * g[4]) - g[1] * (g[1] * g[5] - g[4] * g[2]) + g[2] * (g[1] * g[4] - g[3] * g[2]);
  {
    const double idet = 1.0 / detg;
    gi[0] = (g[3] * g[5] - g[4] * g[4]) * idet;
    gi[1] = (g[2] * g[4] - g[1] * g[5]) * idet;
    gi[2] = (g[1] * g[4] - g[2] * g[3]) * idet;
    gi[3] = (g[0] * g[5] - g[2] * g[2]) * idet;
    gi[4] = (g[1] * g[2] - g[0] * g[4]) * idet;
    gi[5] = (g[0] * g[3] - g[1] * g[1]) * idet;
  }
  const double ichi = 1.0 / chi;
#define G_(i, j) g[sym(i, j)]
#define GI(i, j) gi[sym(i, j)]

  // ---- Christoffels of the conformal metric: Gl[k][ij] = Gamma~_kij, Gu[k][ij] = Gamma~^k_ij
  double Gl[3][6], Gu[3][6], Gt[3];
  {
    double dg[3][6];   // dg[k][ij] = d_k gamma~_ij
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int a = 0; a < 6; ++a) dg[c][a] = d1(GXX + a, c);
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) Gl[c][sym(a, b)] = 0.5 * (dg[a][sym(c, b)] + dg[b][sym(c, a)] - dg[c][sym(a, b)]);
  }
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int a = 0; a < 6; ++a) Gu[c][a] = GI(c, 0) * Gl[0][a] + GI(c, 1) * Gl[1][a] + GI(c, 2) * Gl[2][a];
#pragma unroll
  for (int c = 0; c < 3; ++c)
    Gt[c] = gi[0] * Gu[c][0] + gi[3] * Gu[c][3] + gi[5] * Gu[c][5] + 2.0 * (gi[1] * Gu[c][1] + gi[2] * Gu[c][2] + gi[4] * Gu[c][4]);

  const double Gh[3] = {ld(F(GAMX)), ld(F(GAMY)), ld(F(GAMZ))};
  double Z[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) Z[c] = 0.5 * chi * (Gh[c] - Gt[c]);          // l.132

  // ---- chi R^_ij  (Eq. 23 times chi), accumulated component by component
  double X[6];   // becomes alpha (chi R^_ij + chi R^chi_ij - 8 pi G chi S_ij) - chi D_i D_j alpha
  {
    double dGh[3][3];   // dGh[a][c] = d_a Gamma^^c
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int c = 0; c < 3; ++c) dGh[a][c] = d1(GAMX + c, a);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b) {
        const int ab = sym(a, b);
        double r = 0.0;
        // -1/2 gamma~^mn d_m d_n gamma~_ab
        r -= 0.5 * (gi[0] * d2(GXX + ab, 0, 0) + gi[3] * d2(GXX + ab, 1, 1) + gi[5] * d2(GXX + ab, 2, 2));
        r -= gi[1] * d2(GXX + ab, 0, 1) + gi[2] * d2(GXX + ab, 0, 2) + gi[4] * d2(GXX + ab, 1, 2);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          r += 0.5 * (G_(c, a) * dGh[b][c] + G_(c, b) * dGh[a][c]);           // gamma~_k(i d_j) Gamma^^k
          r += 0.5 * Gh[c] * (Gl[a][sym(b, c)] + Gl[b][sym(a, c)]);           // Gamma^^k Gamma~_(ij)k
        }
#pragma unroll
        for (int m = 0; m < 3; ++m)
#pragma unroll
          for (int n = 0; n < 3; ++n) {
            double t = 0.0;
#pragma unroll
            for (int c = 0; c < 3; ++c)
              t += Gu[c][sym(m, a)] * Gl[b][sym(c, n)] + Gu[c][sym(m, b)] * Gl[a][sym(c, n)] + Gu[c][sym(m, a)] * Gl[c][sym(n, b)];
            r += GI(m, n) * t;
          }
        X[ab] = chi * r;
      }
  }
  double Rtr = 0.0;   // gamma^ij (R_ij + 2 D_(i Z_j)) = gamma~^ij (chi R^_ij + chi R^chi_ij)

  // ---- chi R^chi_ij (Eq. 22), physical Hessian of the lapse (R25), matter (l.188-192, l.260)
  double dchi[3], dal[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) { dchi[a] = d1(CHI, a); dal[a] = d1(ALPHA, a); }
  double gdchi[3];   // gamma~^kl d_l chi
#pragma unroll
  for (int c = 0; c < 3; ++c) gdchi[c] = GI(c, 0) * dchi[0] + GI(c, 1) * dchi[1] + GI(c, 2) * dchi[2];
  double lapal;      // D_i D^i alpha, Eq. (24)
  {
    double ddchi[6], ddal[6];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b) { ddchi[sym(a, b)] = d2(CHI, a, b); ddal[sym(a, b)] = d2(ALPHA, a, b); }
    double lapchi = 0.0, Ghdchi = 0.0, Zl[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      Ghdchi += Gh[a] * dchi[a];
      Zl[a] = G_(a, 0) * Z[0] + G_(a, 1) * Z[1] + G_(a, 2) * Z[2];        // Z^k gamma~_ka
#pragma unroll
      for (int b = 0; b < 3; ++b) lapchi += GI(a, b) * (ddchi[sym(a, b)] - 1.5 * ichi * dchi[a] * dchi[b]);
    }
    lapal = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      lapal -= chi * Gt[a] * dal[a];
#pragma unroll
      for (int b = 0; b < 3; ++b) lapal += chi * GI(a, b) * ddal[sym(a, b)] - 0.5 * GI(a, b) * dal[a] * dchi[b];
    }
    double gdal_chi = 0.0;   // gamma~^kl d_l chi d_k alpha
#pragma unroll
    for (int c = 0; c < 3; ++c) gdal_chi += gdchi[c] * dal[c];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b) {
        const int ab = sym(a, b);
        double c_ = 0.5 * ddchi[ab] - 0.25 * ichi * dchi[a] * dchi[b];
        double Gdal = 0.0;   // Gamma~^k_ab d_k alpha
#pragma unroll
        for (int c = 0; c < 3; ++c) { c_ -= 0.5 * Gu[c][ab] * dchi[c]; Gdal += Gu[c][ab] * dal[c]; }
        c_ += ichi * (Zl[a] * dchi[b] + Zl[b] * dchi[a]);                    // (2/chi) Z^k gamma~_k(i d_j) chi
        c_ += 0.5 * g[ab] * (lapchi - Ghdchi);
        // D_a D_b alpha = dd alpha - Gamma^k_ab d_k alpha, Gamma^k_ab = Gamma~^k_ab - (delta^k_a d_b chi + delta^k_b d_a chi - gamma~_ab gamma~^kl d_l chi)/(2 chi)
        const double DDal = ddal[ab] - Gdal + 0.5 * ichi * (dal[a] * dchi[b] + dal[b] * dchi[a] - g[ab] * gdal_chi);
        const double ric = X[ab] + c_;                                       // chi (R^_ab + R^chi_ab)
        Rtr += (a == b ? 1.0 : 2.0) * gi[ab] * ric;
        X[ab] = al * ric - chi * DDal;
      }
  }
  // ---- matter
  const double G8 = 8.0 * 3.14159265358979323846 * par.grav_G;
  const double isg = chi * sqrt(chi);   // 1/sqrt(gamma)
  double uc[10];
#pragma unroll
  for (int a = 0; a < 10; ++a) uc[a] = ld(F(DBAR + a));
  double Sij[6];   // undensitised S_ij, l.260
  double E, Sl[3], vu[3];
  {
    const double W = ld(P + (size_t)WLOR * sp + pt), pr = ld(P + (size_t)PRESS * sp + pt);
    double vl[3], Bu[3], Bl[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) { vu[a] = ld(P + (size_t)(VX + a) * sp + pt); Bu[a] = uc[6 + a] * isg; Sl[a] = uc[3 + a] * isg; }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      vl[a] = ichi * (G_(a, 0) * vu[0] + G_(a, 1) * vu[1] + G_(a, 2) * vu[2]);
      Bl[a] = ichi * (G_(a, 0) * Bu[0] + G_(a, 1) * Bu[1] + G_(a, 2) * Bu[2]);
    }
    const double B2 = Bu[0] * Bl[0] + Bu[1] * Bl[1] + Bu[2] * Bl[2];
    const double Bv = Bu[0] * vl[0] + Bu[1] * vl[1] + Bu[2] * vl[2];
    const double iW2 = 1.0 / (W * W);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b) {
        const double gab = ichi * g[sym(a, b)];
        Sij[sym(a, b)] = 0.5 * (vl[a] * Sl[b] + vl[b] * Sl[a]) + gab * pr - 0.5 * iW2 * (2.0 * Bl[a] * Bl[b] - gab * B2)
                         - 0.5 * Bv * (Bl[a] * vl[b] + Bl[b] * vl[a] - gab * Bv);
      }
    E = (uc[2] + uc[0]) * isg;   // R6: tau_ADM = tau + D
  }
  double Str = 0.0;   // S = gamma^ij S_ij
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) Str += chi * GI(a, b) * Sij[sym(a, b)];
  {
    double trX = 0.0;
#pragma unroll
    for (int a = 0; a < 6; ++a) X[a] -= al * G8 * chi * Sij[a];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) trX += GI(a, b) * X[sym(a, b)];
#pragma unroll
    for (int a = 0; a < 6; ++a) X[a] -= g[a] * trX * (1.0 / 3.0);            // [..]^TF
  }

  // ---- shift derivatives
  double dbe[3][3];   // dbe[a][c] = d_a beta^c
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int c = 0; c < 3; ++c) dbe[a][c] = d1(BETAX + c, a);
  const double divb = dbe[0][0] + dbe[1][1] + dbe[2][2];

  // ---- curvature fields
  double A[6];
#pragma unroll
  for (int a = 0; a < 6; ++a) A[a] = ld(F(AXX + a));
  const double Kh = ld(F(KHAT)), Th = ld(F(THETA));
  const double Ktot = Kh + 2.0 * Th;
  double Aud[3][3];   // A~^a_b
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) Aud[a][b] = GI(a, 0) * A[sym(0, b)] + GI(a, 1) * A[sym(1, b)] + GI(a, 2) * A[sym(2, b)];
  const double trA = Aud[0][0] + Aud[1][1] + Aud[2][2];                       // R4
  double AA = 0.0;
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) AA += Aud[a][b] * Aud[b][a];
  double Auu[6];      // A~^ab
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = a; b < 3; ++b) Auu[sym(a, b)] = Aud[a][0] * GI(0, b) + Aud[a][1] * GI(1, b) + Aud[a][2] * GI(2, b);

  const double sig = par.sigma_ko_spacetime;
  const double logdet = log(detg);
  // ---- Eq. (13)
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = a; b < 3; ++b) {
      const int ab = sym(a, b);
      double s = adv_ko(F(GXX + ab), st, be, sig);
#pragma unroll
      for (int c = 0; c < 3; ++c) s += G_(a, c) * dbe[b][c] + G_(c, b) * dbe[a][c];
      s += -(2.0 / 3.0) * g[ab] * divb - 2.0 * al * (A[ab] - g[ab] * trA * (1.0 / 3.0)) - al * (1.0 / 3.0) * par.kappa_c * g[ab] * logdet;
      OUT(GXX + ab) = s;
    }
  // ---- Eq. (14)
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = a; b < 3; ++b) {
      const int ab = sym(a, b);
      double s = adv_ko(F(AXX + ab), st, be, sig);
      double AAab = 0.0;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        s += A[sym(a, c)] * dbe[b][c] + A[sym(c, b)] * dbe[a][c];
        AAab += A[sym(a, c)] * Aud[c][b];
      }
      s += -(2.0 / 3.0) * A[ab] * divb - al * (1.0 / 3.0) * par.kappa_c * g[ab] * trA + X[ab] + al * (Kh * A[ab] - 2.0 * AAab);
      OUT(AXX + ab) = s;
    }
  // ---- Eq. (15)
  OUT(CHI) = adv_ko(F(CHI), st, be, sig) + (2.0 / 3.0) * chi * (al * Ktot - divb);
  // ---- Eqs. (16), (17)
  const double Zdal = Z[0] * dal[0] + Z[1] * dal[1] + Z[2] * dal[2];
  OUT(KHAT) = adv_ko(F(KHAT), st, be, sig) - lapal + al * (Ktot * Ktot * (1.0 / 3.0) + AA + 0.5 * G8 * (E + Str) + par.kappa_z * (1.0 - par.kappa_2) * Th) + 2.0 * Zdal;
  OUT(THETA) = adv_ko(F(THETA), st, be, sig) + 0.5 * al * (Rtr + (2.0 / 3.0) * Kh * Kh + (2.0 / 3.0) * Th * (Kh - 2.0 * Th) - AA) - Zdal
               - al * (G8 * E + par.kappa_z * (2.0 + par.kappa_2) * Th);
  // ---- Eqs. (18)-(20)
  {
    double dKh[3], dTh[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) { dKh[a] = d1(KHAT, a); dTh[a] = d1(THETA, a); }
    // second derivatives of the shift, contracted at once: lapb[c] = gamma~^jk d_j d_k beta^c, ddiv[j] = d_j d_k beta^k
    double lapb[3], ddiv[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double dd[6];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) dd[sym(a, b)] = d2(BETAX + c, a, b);
      lapb[c] = gi[0] * dd[0] + gi[3] * dd[3] + gi[5] * dd[5] + 2.0 * (gi[1] * dd[1] + gi[2] * dd[2] + gi[4] * dd[4]);
#pragma unroll
      for (int a = 0; a < 3; ++a) ddiv[a] += dd[sym(a, c)];
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      double s = adv_ko(F(GAMX + a), st, be, sig) + (2.0 / 3.0) * Gh[a] * divb + lapb[a];
      double b1 = 0.0, b2 = 0.0;
#pragma unroll
      for (int b = 0; b < 3; ++b) {
        s += -Gh[b] * dbe[b][a] + GI(a, b) * ddiv[b] * (1.0 / 3.0) - 2.0 * Auu[sym(a, b)] * dal[b];
#pragma unroll
        for (int c = 0; c < 3; ++c) b1 += Gu[a][sym(b, c)] * Auu[sym(b, c)];
        b1 += -1.5 * ichi * Auu[sym(a, b)] * dchi[b] - (2.0 / 3.0) * GI(a, b) * dKh[b] - G8 * GI(a, b) * Sl[b];
        b2 -= GI(a, b) * (dTh[b] * (1.0 / 3.0) + Th / al * dal[b]);
      }
      b2 -= Z[a] * ichi * (par.kappa_z + (2.0 / 3.0) * Ktot);
      OUT(GAMX + a) = s + 2.0 * al * (b1 + b2);
    }
  }
  // ---- gauge, Eqs. (25)-(26)
  OUT(ALPHA) = adv_ko(F(ALPHA), st, be, sig) - 2.0 * al * par.f_alpha * Kh;
#pragma unroll
  for (int a = 0; a < 3; ++a) OUT(BETAX + a) = adv_ko(F(BETAX + a), st, be, sig) + 0.75 * par.f_beta * Gh[a] - par.eta_shift * (be[a] - par.beta0[a]);

  // ---- sources of the GRMHD system (right-hand sides of Eq. 32); the flux divergence is subtracted by flux.cu
  {
    const double sg = 1.0 / isg;
    // Sbar^ab = sqrt(gamma) chi^2 gamma~^ac gamma~^bd S_cd ; tr Sbar = sqrt(gamma) S
    double Suu[6];
    {
      double T[3][3];   // gamma~^ac S_cb
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) T[a][b] = GI(a, 0) * Sij[sym(0, b)] + GI(a, 1) * Sij[sym(1, b)] + GI(a, 2) * Sij[sym(2, b)];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) Suu[sym(a, b)] = sg * chi * chi * (T[a][0] * GI(0, b) + T[a][1] * GI(1, b) + T[a][2] * GI(2, b));
    }
    const double trS = sg * Str;
    double stau = al * (1.0 / 3.0) * trS * Ktot;
    double SA = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) SA += Suu[sym(a, b)] * A[sym(a, b)];
    stau += al * ichi * SA;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double Sup = chi * (GI(a, 0) * uc[3] + GI(a, 1) * uc[4] + GI(a, 2) * uc[5]);   // Sbar^a
      stau -= Sup * dal[a];
    }
    OUT(DBAR) = 0.0;
    OUT(DYEBAR) = 0.0;
    OUT(TAUBAR) = stau;
    const double cb2 = par.c_b * par.c_b;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      double s = -(uc[2] + uc[0]) * dal[a] - 0.5 * al * ichi * trS * dchi[a];
      double Sdg = 0.0;   // Sbar^jk d_a gamma~_jk, with d_a gamma~_jk = Gamma~_jak + Gamma~_kaj
#pragma unroll
      for (int b = 0; b < 3; ++b) {
        s += uc[3 + b] * dbe[a][b];
#pragma unroll
        for (int c = 0; c < 3; ++c) Sdg += Suu[sym(b, c)] * (Gl[b][sym(a, c)] + Gl[c][sym(a, b)]);
      }
      OUT(SXBAR + a) = s + 0.5 * al * ichi * Sdg;
      double sb = -al * (chi * Gh[a] - 2.0 * Z[a]);
#pragma unroll
      for (int c = 0; c < 3; ++c) sb += GI(c, a) * (-0.5 * al * dchi[c] + chi / cb2 * dal[c]);
      OUT(BXBAR + a) = uc[9] * sb;
    }
    OUT(PHIBAR) = -al * cb2 * uc[9] * Ktot - al * par.kappa_b * uc[9] + cb2 * (uc[6] * dal[0] + uc[7] * dal[1] + uc[8] * dal[2]);
    if (par.sigma_ko_matter != 0.0) {                                        // R16: optional KO on the matter fields
      const double zero[3] = {0.0, 0.0, 0.0};
#pragma unroll 1
      for (int a = 0; a < 10; ++a) OUT(DBAR + a) += adv_ko(F(DBAR + a), st, zero, par.sigma_ko_matter);
    }
  }
#undef G_
#undef GI
}

cudaError_t launch_rhs_ccz4(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* K, size_t sk, cudaStream_t s) {
  dim3 block(32, 4, 2);
  dim3 grid((d.nx + block.x - 1) / block.x, (d.ny + block.y - 1) / block.y, (d.nz + block.z - 1) / block.z);
  k_rhs_ccz4<<<grid, block, 0, s>>>(d, par, U, su, P, sp, K, sk);
  return cudaGetLastError();
}

}  // namespace mhd
