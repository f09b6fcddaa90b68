// a10-a12: grey M1 neutrino transport, 3 species (Sec. II C, III D, App. B, App. C).
//   k_m1_point     every grid point, every species: Minerbo closure (root of Eq. 50 for xi with Eqs. 42-49), then the flux
//                  brackets of Eqs. (38)-(40) in the three directions, the speed bound (B4)-(B5, reading R32), the
//                  opacity sum kappa_a + kappa_s and P_ij, written to the M1 work slot (25 fields per species).
//   k_m1_div       every interior zone: flux-limited advection-diffusion fluxes of Sec. III D (Eqs. 77-78, readings R20) at
//                  the two x faces from the work slot, the geometric sources of Eqs. (39)-(40) (reading R19) -> KV.
//   k_m1_march     the y and z faces as a march (register window along the line), added to KV.
//   k_m1_implicit  every grid point: the pointwise implicit solve of App. C — closure frozen at V* (R21), Newton on the
//                  4x4 system (C13)-(C16) with the Jacobian (C28)-(C35), N from (C11); writes V^(i) and the stiff source R.
//   k_m1_backreact K_fluid -= sum over species of R (l.256, l.312-316; R24).
// One thread per point; x-contiguous warps (coalesced field loads). The closure solve is a bounded Brent iteration.
#include "mhd_internal.cuh"
#include "rootfind.cuh"

namespace mhd {

namespace {

constexpr int M1W = 25;   // work fields per species: 3 x (5 fluxes + speed) = 18, kappa = 1, P_ij = 6

struct Geo {   // geometry and fluid state at one point
  double al, be[3], chi, sg, gl[6], gu[6], vu[3], W, rho, T;
};
__device__ __forceinline__ constexpr int sy(int i, int j) { return i <= j ? (i * (5 - i)) / 2 + j : (j * (5 - j)) / 2 + i; }

__device__ __forceinline__ void load_geo(const double* __restrict__ U, size_t su, const double* __restrict__ P, size_t sp, size_t pt, Geo& q) {
  double g[6];
#pragma unroll
  for (int a = 0; a < 6; ++a) g[a] = __ldg(U + (size_t)(GXX + a) * su + pt);
  q.chi = __ldg(U + (size_t)CHI * su + pt);
  const double det = g[0] * (g[3] * g[5] - g[4] * g[4]) - g[1] * (g[1] * g[5] - g[4] * g[2]) + g[2] * (g[1] * g[4] - g[3] * g[2]);
  const double f = q.chi / det, ichi = 1.0 / q.chi;
  q.gu[0] = (g[3] * g[5] - g[4] * g[4]) * f;
  q.gu[1] = (g[2] * g[4] - g[1] * g[5]) * f;
  q.gu[2] = (g[1] * g[4] - g[2] * g[3]) * f;
  q.gu[3] = (g[0] * g[5] - g[2] * g[2]) * f;
  q.gu[4] = (g[1] * g[2] - g[0] * g[4]) * f;
  q.gu[5] = (g[0] * g[3] - g[1] * g[1]) * f;
#pragma unroll
  for (int a = 0; a < 6; ++a) q.gl[a] = g[a] * ichi;
  q.sg = 1.0 / (q.chi * sqrt(q.chi));
  q.al = __ldg(U + (size_t)ALPHA * su + pt);
#pragma unroll
  for (int i = 0; i < 3; ++i) { q.be[i] = __ldg(U + (size_t)(BETAX + i) * su + pt); q.vu[i] = __ldg(P + (size_t)(VX + i) * sp + pt); }
  q.W = __ldg(P + (size_t)WLOR * sp + pt);
  q.rho = __ldg(P + (size_t)RHO * sp + pt);
  q.T = __ldg(P + (size_t)TEMP * sp + pt);
}
__device__ __forceinline__ void mul_sym(const double m[6], const double a[3], double o[3]) {
#pragma unroll
  for (int i = 0; i < 3; ++i) o[i] = m[sy(i, 0)] * a[0] + m[sy(i, 1)] * a[1] + m[sy(i, 2)] * a[2];
}
__device__ __forceinline__ double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

struct Closure { double xi, chi, J, Hn, H[3], P[6]; };

// Eqs. (42)-(48) for a given Eddington factor
__device__ __forceinline__ void moments(double chiE, double E, const double F[3], const double Fu[3], double iF2, const double vu[3],
                                        const double vl[3], double W, const double gl[6], Closure& c) {
  const double dthin = 0.5 * (3.0 * chiE - 1.0), dthick = 1.5 * (1.0 - chiE);
  const double W2 = W * W, i2w = 1.0 / (2.0 * W2 + 1.0);
  const double Fv = dot3(vu, F);
  const double Jthick = 3.0 * i2w * ((2.0 * W2 - 1.0) * E - 2.0 * W2 * Fv);                            // Eq. (47)
  double Htu[3], Ht[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) Htu[i] = Fu[i] / W + W * vu[i] * i2w * ((4.0 * W2 + 1.0) * Fv - 4.0 * W2 * E);
  mul_sym(gl, Htu, Ht);
  double Pvv = 0.0, Pv[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) {
      const double thin = E * F[i] * F[j] * iF2;                                                       // Eq. (45)
      const double thick = (4.0 / 3.0) * Jthick * W2 * vl[i] * vl[j] + W * (Ht[i] * vl[j] + Ht[j] * vl[i]) + Jthick * gl[sy(i, j)] * (1.0 / 3.0);
      const double p = dthin * thin + dthick * thick;                                                  // Eq. (48)
      c.P[sy(i, j)] = p;
      Pvv += (i == j ? 1.0 : 2.0) * p * vu[i] * vu[j];
      Pv[i] += p * vu[j];
      if (i != j) Pv[j] += p * vu[i];
    }
  c.J = W2 * (E - 2.0 * Fv + Pvv);                                                                      // Eq. (42)
  c.Hn = W * (c.J - E + Fv);                                                                            // Eq. (43)
#pragma unroll
  for (int i = 0; i < 3; ++i) c.H[i] = W * (F[i] - Pv[i] - c.J * vl[i]);                                // Eq. (44)
  c.chi = chiE;
}
__device__ __forceinline__ double eddington(double xi) { return 1.0 / 3.0 + xi * xi * (6.0 - 2.0 * xi + 6.0 * xi * xi) * (1.0 / 15.0); }

// root of Eq. (50) on [0, 1]
__device__ void closure_solve(double E, const double F[3], const Geo& q, Closure& c) {
  double Fu[3], vl[3];
  mul_sym(q.gu, F, Fu);
  mul_sym(q.gl, q.vu, vl);
  const double F2 = dot3(Fu, F);
  const double iF2 = F2 < 1e-30 * E * E ? 0.0 : 1.0 / F2;                                                       // R22
  const double iE2 = 1.0 / (E * E);
  auto R = [&](double xi) {
    moments(eddington(xi), E, F, Fu, iF2, q.vu, vl, q.W, q.gl, c);
    double Hu[3];
    mul_sym(q.gu, c.H, Hu);
    return (xi * xi * c.J * c.J - (dot3(Hu, c.H) - c.Hn * c.Hn)) * iE2;
  };
  const double R0 = R(0.0);
  if (R0 >= 0.0) { c.xi = 0.0; return; }
  const double R1 = R(1.0);
  if (R1 <= 0.0) { c.xi = 1.0; return; }
  // R(0) < 0 < R(1). For a fluid at rest xi = |F| / E exactly, for a moving one it is off by O(v): one evaluation there
  // shrinks the bracket from [0, 1] to one side of it before Brent starts.
  bool ok;
  double a = 0.0, b = 1.0, Ra = R0, Rb = R1;
  const double xg = sqrt(F2) / E;
  if (xg > 0.0 && xg < 1.0) {
    const double Rg = R(xg);
    if (Rg == 0.0) { c.xi = xg; return; }
    if (Rg < 0.0) { a = xg; Ra = Rg; } else { b = xg; Rb = Rg; }
  }
  c.xi = brent_root(R, a, b, Ra, Rb, 100, ok);
  R(c.xi);
}

__device__ __forceinline__ void opacities(const Par& par, int s, double rho, double T, double& ka, double& ks, double& eta) {
  const double x = rho / par.m1_rho0;
  ka = par.m1_kappa0 * x * x * par.m1_species_scale[s];
  ks = ka;
  const double T2 = T * T;
  eta = par.m1_arad * ka * T2 * T2;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128, 3) k_m1_point(const __grid_constant__ Dims d, const __grid_constant__ Par par, const double* __restrict__ U, size_t su,
                                                  const double* __restrict__ P, size_t sp, const double* __restrict__ V, size_t sv,
                                                  double* __restrict__ Wk, size_t sw) {
  const long long pt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (pt >= d.npts) return;
  Geo q;
  load_geo(U, su, P, sp, pt, q);
  const double isg = 1.0 / q.sg;
#pragma unroll 1
  for (int s = 0; s < 3; ++s) {
    double u[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) u[f] = __ldg(V + (size_t)(5 * s + f) * sv + pt);
    const double E = u[1] * isg, F[3] = {u[2] * isg, u[3] * isg, u[4] * isg};
    Closure c;
    closure_solve(E, F, q, c);
    double Fu[3], Hu[3];
    mul_sym(q.gu, F, Fu);
    mul_sym(q.gu, c.H, Hu);
#pragma unroll
    for (int i = 0; i < 3; ++i) Hu[i] += c.Hn * q.be[i] / q.al;                                          // H^i (l.326)
    const double Fv = dot3(q.vu, F);
    const double iGam = c.J / (q.W * (E - Fv));
    const double F2 = dot3(Fu, F), W2 = q.W * q.W;
    double ka, ks, eta;
    opacities(par, s, q.rho, q.T, ka, ks, eta);
    double* out = Wk + (size_t)(M1W * s) * sw + pt;
#pragma unroll
    for (int dir = 0; dir < 3; ++dir) {
      double* o = out + (size_t)(6 * dir) * sw;
      o[0] = (-q.W * q.be[dir] + q.al * q.W * q.vu[dir] + q.al * Hu[dir] / c.J) * u[0] * iGam;             // Eq. (38)
      o[sw] = -q.be[dir] * u[1] + q.al * q.sg * Fu[dir];                                                  // Eq. (39)
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        const double Pid = q.gu[sy(dir, 0)] * c.P[sy(i, 0)] + q.gu[sy(dir, 1)] * c.P[sy(i, 1)] + q.gu[sy(dir, 2)] * c.P[sy(i, 2)];
        o[(2 + i) * sw] = -q.be[dir] * u[2 + i] + q.al * q.sg * Pid;                                      // Eq. (40)
      }
      const double gdd = q.gu[sy(dir, dir)];
      double thin = fabs(q.be[dir]);
      if (F2 >= 1e-30 * E * E) thin += q.al * fmin(fmax(fabs(Fu[dir]) / sqrt(F2), E * fabs(Fu[dir]) / F2), sqrt(gdd));   // (B5), R32
      const double thick = fabs(q.be[dir]) + q.al * fmax((2.0 * W2 * fabs(q.vu[dir]) + sqrt(fmax((2.0 * W2 + 1.0) * gdd - 2.0 * W2 * q.vu[dir] * q.vu[dir], 0.0))) / (2.0 * W2 + 1.0),
                                                         fabs(q.vu[dir]));
      o[5 * sw] = 0.5 * (3.0 * c.chi - 1.0) * thin + 1.5 * (1.0 - c.chi) * thick;                         // (B4)
    }
    out[18 * sw] = ka + ks;
#pragma unroll
    for (int a = 0; a < 6; ++a) out[(19 + a) * sw] = c.P[a];
  }
}

// ---------------------------------------------------------------------------------------------------------------
namespace {
// F^_{i+1/2} of Eq. (77) from u_{i-1..i+2}, the fluxes at i, i+1, lambda_{i+1/2} and A_{i+1/2}
// min / max as plain selects: fmin / fmax carry IEEE NaN handling that costs six instructions each on sm_100a (no FP64 min/max instruction), and the face
// formula below is mostly min / max; the operands here are never NaN where the result is used
__device__ __forceinline__ double tmin(double a, double b) { return b < a ? b : a; }
__device__ __forceinline__ double tmax(double a, double b) { return a < b ? b : a; }
__device__ __forceinline__ double m1_face(double um, double u0, double up, double upp, double F0, double F1, double lam, double A0, double oe) {
  const double dm = u0 - um, d0 = up - u0, dp = upp - up;
  const double r2 = 2.0 / d0;                                                                           // one reciprocal per face and field
  const double Phi = d0 == 0.0 ? 1.0 : tmax(0.0, tmin(1.0, tmin(dm * r2, dp * r2)));                    // Eq. (78), R20
  const double tiny = oe * tmax(tmax(fabs(um), fabs(u0)), tmax(fabs(up), fabs(upp)));                   // R33 (oe = 0: the printed rule; oe < 0: switch off)
  // l.565-570; min(|dm|, |d0|, |dp|) > tiny as three chained compares
  const double A = (oe >= 0.0 && dm * d0 < 0.0 && d0 * dp < 0.0 && fabs(dm) > tiny && fabs(d0) > tiny && fabs(dp) > tiny) ? 1.0 : A0;
  const double FHO = 0.5 * (F0 + F1);
  return FHO - A * (1.0 - Phi) * (0.5 * lam * d0);                                                      // F^HO - F^LO = lambda d0 / 2
}
__device__ __forceinline__ double d1c(const double* __restrict__ u, long long s, double i12h) {
  return (8.0 * (__ldg(u + s) - __ldg(u - s)) - (__ldg(u + 2 * s) - __ldg(u - 2 * s))) * i12h;
}
}  // namespace

__global__ void __launch_bounds__(128, 3) k_m1_div(const __grid_constant__ Dims d, double oe, const double* __restrict__ U, size_t su,
                                                const double* __restrict__ V, size_t sv, const double* __restrict__ Wk, size_t sw,
                                                double* __restrict__ KV, size_t sk) {
  // a CTA owns a 16 x 4 x 2 block of zones: the y / z neighbours of the metric derivatives below are then mostly loaded by the same CTA (L1 hits)
  const int i = blockIdx.x * 16 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y, k = blockIdx.z * 2 + threadIdx.z;
  if (i >= d.nx || j >= d.ny || k >= d.nz) return;
  const size_t pt = (size_t)(k + d.ng) * d.sz + (size_t)(j + d.ng) * d.sy + (i + d.ng);
  const long long st[3] = {1, d.sy, d.sz};
  const double h[3] = {d.dx, d.dy, d.dz};
  // the pressure tensors the source terms of the second species loop read are pulled into L1 now (three exposed HBM round trips otherwise)
#pragma unroll
  for (int s = 0; s < 3; ++s)
#pragma unroll
    for (int a = 0; a < 6; ++a) asm volatile("prefetch.global.L1 [%0];" ::"l"(Wk + (size_t)(M1W * s + 19 + a) * sw + pt));
#pragma unroll 1
  for (int s = 0; s < 3; ++s) {
    double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    const double* wk = Wk + (size_t)(M1W * s) * sw + pt;
    {                                                  // x faces here; the y and z faces are added by k_m1_march
      constexpr int dir = 0;
      const long long ls = st[dir];
      const double* wl = wk + (size_t)(6 * dir + 5) * sw;
      const double* wkap = wk + (size_t)18 * sw;
      const double lm = __ldg(wl - ls), l0 = __ldg(wl), lp = __ldg(wl + ls);
      const double km = __ldg(wkap - ls), k0 = __ldg(wkap), kp = __ldg(wkap + ls);
      const double lamL = fmax(lm, l0), lamR = fmax(l0, lp);
      const double khL = 0.5 * (km + k0) * h[dir], khR = 0.5 * (k0 + kp) * h[dir];
      // tanh(x) rounds to 1 in FP64 for x >= 20: optically thin faces skip the evaluation
      const double AL = khL > 0.05 ? tanh(1.0 / khL) : 1.0, AR = khR > 0.05 ? tanh(1.0 / khR) : 1.0;
      const double ih = 1.0 / h[dir];
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        const double* u = V + (size_t)(5 * s + f) * sv + pt;
        const double* F = wk + (size_t)(6 * dir + f) * sw;
        const double u2m = __ldg(u - 2 * ls), um = __ldg(u - ls), u0 = __ldg(u), up = __ldg(u + ls), u2p = __ldg(u + 2 * ls);
        const double Fm = __ldg(F - ls), F0 = __ldg(F), Fp = __ldg(F + ls);
        const double fR = m1_face(um, u0, up, u2p, F0, Fp, lamR, AR, oe);
        const double fL = m1_face(u2m, um, u0, up, Fm, F0, lamL, AL, oe);
        acc[f] -= (fR - fL) * ih;
      }
    }
#pragma unroll
    for (int f = 0; f < 5; ++f) KV[(size_t)(5 * s + f) * sk + pt] = acc[f];
  }
  // ---- geometry for the sources of Eqs. (39)-(40)
  double g[6], gu[6], dg[3][6], dchi[3], dal[3], dbe[3][3], At[6], be[3];
#pragma unroll
  for (int a = 0; a < 6; ++a) { g[a] = __ldg(U + (size_t)(GXX + a) * su + pt); At[a] = __ldg(U + (size_t)(AXX + a) * su + pt); }
  const double chi = __ldg(U + (size_t)CHI * su + pt), al = __ldg(U + (size_t)ALPHA * su + pt);
  const double Ktot = __ldg(U + (size_t)KHAT * su + pt) + 2.0 * __ldg(U + (size_t)THETA * su + pt);
  {
    const double det = g[0] * (g[3] * g[5] - g[4] * g[4]) - g[1] * (g[1] * g[5] - g[4] * g[2]) + g[2] * (g[1] * g[4] - g[3] * g[2]);
    const double f = chi / det;
    gu[0] = (g[3] * g[5] - g[4] * g[4]) * f; gu[1] = (g[2] * g[4] - g[1] * g[5]) * f; gu[2] = (g[1] * g[4] - g[2] * g[3]) * f;
    gu[3] = (g[0] * g[5] - g[2] * g[2]) * f; gu[4] = (g[1] * g[2] - g[0] * g[4]) * f; gu[5] = (g[0] * g[3] - g[1] * g[1]) * f;
  }
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const double i12h = 1.0 / (12.0 * h[k]);
#pragma unroll
    for (int a = 0; a < 6; ++a) dg[k][a] = d1c(U + (size_t)(GXX + a) * su + pt, st[k], i12h);
    dchi[k] = d1c(U + (size_t)CHI * su + pt, st[k], i12h);
    dal[k] = d1c(U + (size_t)ALPHA * su + pt, st[k], i12h);
#pragma unroll
    for (int c = 0; c < 3; ++c) dbe[k][c] = d1c(U + (size_t)(BETAX + c) * su + pt, st[k], i12h);
    be[k] = 0.0;
  }
  (void)be;
  const double sg = 1.0 / (chi * sqrt(chi)), ichi = 1.0 / chi;
#pragma unroll 1
  for (int s = 0; s < 3; ++s) {
    const double* wk = Wk + (size_t)(M1W * s) * sw + pt;
    double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    double kold[5];                                      // flux part written above by this thread: fetched before the arithmetic
#pragma unroll
    for (int f = 1; f < 5; ++f) kold[f] = KV[(size_t)(5 * s + f) * sk + pt];
    // ---- geometric sources
    double Pl[6], ub[5];
#pragma unroll
    for (int a = 0; a < 6; ++a) Pl[a] = __ldg(wk + (size_t)(19 + a) * sw);
#pragma unroll
    for (int f = 0; f < 5; ++f) ub[f] = __ldg(V + (size_t)(5 * s + f) * sv + pt);
    double T[3][3], Puu[6];   // T = gamma^ik P_kj ; Pbar^ij = sqrt(gamma) gamma^ik gamma^jl P_kl
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) T[a][b] = gu[sy(a, 0)] * Pl[sy(0, b)] + gu[sy(a, 1)] * Pl[sy(1, b)] + gu[sy(a, 2)] * Pl[sy(2, b)];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b) Puu[sy(a, b)] = sg * (T[a][0] * gu[sy(0, b)] + T[a][1] * gu[sy(1, b)] + T[a][2] * gu[sy(2, b)]);
    double trP = 0.0, PA = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) { trP += ichi * g[sy(a, b)] * Puu[sy(a, b)]; PA += Puu[sy(a, b)] * At[sy(a, b)]; }
    double sE = al * (1.0 / 3.0) * trP * Ktot + al * ichi * PA;                                          // R19
#pragma unroll
    for (int a = 0; a < 3; ++a) sE -= (gu[sy(a, 0)] * ub[2] + gu[sy(a, 1)] * ub[3] + gu[sy(a, 2)] * ub[4]) * dal[a];
    acc[1] += sE;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      double sF = -ub[1] * dal[a] - 0.5 * al * ichi * trP * dchi[a];
      double Pdg = 0.0;
#pragma unroll
      for (int b = 0; b < 3; ++b) {
        sF += ub[2 + b] * dbe[a][b];
#pragma unroll
        for (int c = 0; c < 3; ++c) Pdg += Puu[sy(b, c)] * dg[a][sy(b, c)];
      }
      acc[2 + a] += sF + 0.5 * al * ichi * Pdg;
    }
#pragma unroll
    for (int f = 1; f < 5; ++f) KV[(size_t)(5 * s + f) * sk + pt] = kold[f] + acc[f];
  }
}

// ---------------------------------------------------------------------------------------------------------------
namespace {
struct AppC {   // quantities of App. C that do not change during the Newton iteration
  double vl[3], v2, W, W2, dthin, dthick;
};
// (C17)-(C27): J, H_i ; also returns f^_i, f^^i, v.f^, 1/|F|
__device__ __forceinline__ void appc_JH(const AppC& a, const Geo& q, double E, const double F[3], double& J, double H[3],
                                        double fh[3], double fhu[3], double& vf, double& iF) {
  double Fu[3];
  mul_sym(q.gu, F, Fu);
  const double F2 = dot3(Fu, F);
  iF = F2 < 1e-30 * E * E ? 0.0 : 1.0 / sqrt(F2);
#pragma unroll
  for (int i = 0; i < 3; ++i) { fh[i] = F[i] * iF; fhu[i] = Fu[i] * iF; }
  vf = dot3(q.vu, fh);
  const double vF = dot3(q.vu, F), W = a.W, W2 = a.W2, i2w = 1.0 / (2.0 * W2 + 1.0);
  const double B0 = W2 * (E - 2.0 * vF);
  const double Bthin = W2 * E * vf * vf;
  const double Bthick = (W2 - 1.0) * i2w * (4.0 * W2 * vF + (3.0 - 2.0 * W2) * E);
  const double avthick = W * Bthick + W * i2w * ((2.0 * W2 - 1.0) * vF + (3.0 - 2.0 * W2) * E);
  const double afthin = W * E * vf;
  J = B0 + a.dthin * Bthin + a.dthick * Bthick;
  const double cv = W * B0 + a.dthin * W * Bthin + a.dthick * avthick, cF = -W + a.dthick * W * a.v2;
#pragma unroll
  for (int i = 0; i < 3; ++i) H[i] = -cv * a.vl[i] - a.dthin * afthin * fh[i] - cF * F[i];
}
// alpha (S_n, S_i), l.312-316
__device__ __forceinline__ void stiff(const AppC& a, const Geo& q, double E, const double F[3], double ka, double ks, double eta,
                                      double S[4], double& J, double fh[3], double fhu[3], double& vf, double& iF) {
  double H[3];
  appc_JH(a, q, E, F, J, H, fh, fhu, vf, iF);
  const double Fv = dot3(q.vu, F);
  S[0] = q.al * a.W * ((eta + ks * J) - (ka + ks) * (E - Fv));
#pragma unroll
  for (int i = 0; i < 3; ++i) S[1 + i] = q.al * (a.W * (eta - ka * J) * a.vl[i] - (ka + ks) * H[i]);
}
__device__ __forceinline__ bool fixup(double efloor, double& E, double F[3], const double gu[6]) {
  bool ch = false;
  if (!(E >= efloor)) { E = efloor; ch = true; }
  double Fu[3];
  mul_sym(gu, F, Fu);
  const double F2 = dot3(Fu, F);
  if (F2 > E * E) { const double s = E / sqrt(F2); F[0] *= s; F[1] *= s; F[2] *= s; ch = true; }
  return ch;
}
__device__ __forceinline__ bool solve4(double A[4][4], double b[4]) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    int p = c;
#pragma unroll
    for (int r = c + 1; r < 4; ++r) if (fabs(A[r][c]) > fabs(A[p][c])) p = r;
    if (A[p][c] == 0.0) return false;
    if (p != c) {
#pragma unroll
      for (int k = 0; k < 4; ++k) { const double t = A[p][k]; A[p][k] = A[c][k]; A[c][k] = t; }
      const double t = b[p]; b[p] = b[c]; b[c] = t;
    }
    const double ip = 1.0 / A[c][c];
#pragma unroll
    for (int r = c + 1; r < 4; ++r) {
      const double f = A[r][c] * ip;
#pragma unroll
      for (int k = c; k < 4; ++k) A[r][k] -= f * A[c][k];
      b[r] -= f * b[c];
    }
  }
#pragma unroll
  for (int r = 3; r >= 0; --r) {
    double s = b[r];
#pragma unroll
    for (int k = r + 1; k < 4; ++k) s -= A[r][k] * b[k];
    b[r] = s / A[r][r];
  }
  return true;
}
}  // namespace

__global__ void __launch_bounds__(128, 3) k_m1_implicit(const __grid_constant__ Dims d, const __grid_constant__ Par par, const double* __restrict__ U, size_t su,
                                                     const double* __restrict__ P, size_t sp, double* __restrict__ V, size_t sv,
                                                     double* __restrict__ R, size_t sr, double adt, uint8_t* __restrict__ flags) {
  const long long pt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (pt >= d.npts) return;
  Geo q;
  load_geo(U, su, P, sp, pt, q);
  const double isg = 1.0 / q.sg;
  AppC a;
  mul_sym(q.gl, q.vu, a.vl);
  a.v2 = dot3(q.vu, a.vl); a.W = q.W; a.W2 = q.W * q.W;
  unsigned flag = 0;
#pragma unroll 1
  for (int s = 0; s < 3; ++s) {
    double ka, ks, eta;
    opacities(par, s, q.rho, q.T, ka, ks, eta);                     // fixed during the solve
    const double Ns = V[(size_t)(5 * s) * sv + pt] * isg;
    double Es = V[(size_t)(5 * s + 1) * sv + pt] * isg;
    double Fs[3] = {V[(size_t)(5 * s + 2) * sv + pt] * isg, V[(size_t)(5 * s + 3) * sv + pt] * isg, V[(size_t)(5 * s + 4) * sv + pt] * isg};
    if (fixup(par.m1_efloor, Es, Fs, q.gu)) flag |= MHD_FLAG_M1FIX;
    {
      Closure c;
      closure_solve(Es, Fs, q, c);                                  // R21: closure from V*, frozen
      a.dthin = 0.5 * (3.0 * c.chi - 1.0); a.dthick = 1.5 * (1.0 - c.chi);
    }
    double E = Es, F[3] = {Fs[0], Fs[1], Fs[2]}, J, S[4], fh[3], fhu[3], vf, iF;
    bool conv = adt == 0.0;
    for (int it = 0; it < par.m1_maxit && !conv; ++it) {
      stiff(a, q, E, F, ka, ks, eta, S, J, fh, fhu, vf, iF);
      double G[4] = {E - Es - adt * S[0], F[0] - Fs[0] - adt * S[1], F[1] - Fs[1] - adt * S[2], F[2] - Fs[2] - adt * S[3]};   // (C13)-(C14)
      const double gn = fmax(fmax(fabs(G[0]), fabs(G[1])), fmax(fabs(G[2]), fabs(G[3])));
      if (gn <= par.m1_tol * (fmax(Es, par.m1_efloor) + adt * q.al * a.W * (eta + (ka + ks) * fmax(Es, E)))) { conv = true; break; }   // R21
      // Jacobian (C28)-(C35)
      const double W = a.W, W2 = a.W2, W3 = W2 * W, kas = ka + ks, i2w = 1.0 / (1.0 + 2.0 * W2);
      const double dJdE = W2 + a.dthin * vf * vf * W2 + a.dthick * (3.0 - 2.0 * W2) * (W2 - 1.0) * i2w;
      const double cJ = 2.0 * W2 * (-1.0 + a.dthin * E * vf * iF + 2.0 * a.dthick * (W2 - 1.0) * i2w);
      const double cJf = -2.0 * a.dthin * W2 * E * vf * vf * iF;
      const double cHE = W3 * (-1.0 - a.dthin * vf * vf + a.dthick * (2.0 * W2 - 3.0) * i2w);
      const double cd = W * (1.0 - a.dthin * E * vf * iF - a.dthick * a.v2);
      const double cvv = 2.0 * W3 * (1.0 - a.dthin * E * vf * iF - a.dthick * (a.v2 + 1.0 / (2.0 * W2 * (1.0 + 2.0 * W2))));
      const double cff = 2.0 * a.dthin * W * E * vf * iF, cvf = 2.0 * a.dthin * W3 * E * vf * vf * iF, cfv = -a.dthin * W * E * iF;
      double M[4][4];
      M[0][0] = 1.0 + adt * q.al * W * (kas - ks * dJdE);
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        const double dJdF = cJ * q.vu[j] + cJf * fhu[j];
        M[0][1 + j] = -adt * q.al * W * (ks * dJdF + kas * q.vu[j]);
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          const double dHdF = cd * (i == j ? 1.0 : 0.0) + cvv * a.vl[i] * q.vu[j] + cff * fh[i] * fhu[j] + cvf * a.vl[i] * fhu[j] + cfv * fh[i] * q.vu[j];
          M[1 + i][1 + j] = (i == j ? 1.0 : 0.0) + adt * q.al * (kas * dHdF + W * ka * a.vl[i] * dJdF);
        }
      }
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        const double dHdE = cHE * a.vl[i] - a.dthin * W * vf * fh[i];
        M[1 + i][0] = adt * q.al * (kas * dHdE + W * ka * dJdE * a.vl[i]);
      }
      if (!solve4(M, G)) break;
      E -= G[0]; F[0] -= G[1]; F[1] -= G[2]; F[2] -= G[3];                                                // (C15)
    }
    if (!conv) flag |= MHD_FLAG_NOCONV;
    if (fixup(par.m1_efloor, E, F, q.gu)) flag |= MHD_FLAG_M1FIX;
    stiff(a, q, E, F, ka, ks, eta, S, J, fh, fhu, vf, iF);
    const double Gam = q.W * (E - dot3(q.vu, F)) / J;                                                     // (C12)
    const double N = (Ns + adt * q.al * eta) / (1.0 + adt * q.al * ka / Gam);                             // (C11), synthetic eta^0 = eta, kappa^0 = kappa_a
    V[(size_t)(5 * s) * sv + pt] = q.sg * N;
    V[(size_t)(5 * s + 1) * sv + pt] = q.sg * E;
    R[(size_t)(5 * s) * sr + pt] = q.sg * q.al * (eta - ka * N / Gam);                                     // Eq. (41)
    R[(size_t)(5 * s + 1) * sr + pt] = q.sg * S[0];
#pragma unroll
    for (int i = 0; i < 3; ++i) { V[(size_t)(5 * s + 2 + i) * sv + pt] = q.sg * F[i]; R[(size_t)(5 * s + 2 + i) * sr + pt] = q.sg * S[1 + i]; }
  }
  if (flag) flags[pt] |= (uint8_t)flag;
}

__global__ void __launch_bounds__(128) k_m1_backreact(const __grid_constant__ Dims d, double mb, const double* __restrict__ R, size_t sr,
                                                      double* __restrict__ K, size_t sk) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.nx) return;
  const size_t pt = (size_t)(blockIdx.z + d.ng) * d.sz + (size_t)(blockIdx.y + d.ng) * d.sy + (i + d.ng);
  double st = 0.0, sS[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    st += __ldg(R + (size_t)(5 * s + 1) * sr + pt);
#pragma unroll
    for (int a = 0; a < 3; ++a) sS[a] += __ldg(R + (size_t)(5 * s + 2 + a) * sr + pt);
  }
  K[(size_t)TAUBAR * sk + pt] -= st;
#pragma unroll
  for (int a = 0; a < 3; ++a) K[(size_t)(SXBAR + a) * sk + pt] -= sS[a];
  K[(size_t)DYEBAR * sk + pt] -= mb * (__ldg(R + pt) - __ldg(R + (size_t)5 * sr + pt));
}

// y / z faces of Eq. (77) as a march: thread = (x column, segment of SEG zones along the line), every node value loaded once per
// segment into a register window; KV (written by k_m1_div with the x faces and the sources) is read-modify-write, fetched early.
template <int DIR, int SEG>
__global__ void __launch_bounds__(128, 4) k_m1_march(const __grid_constant__ Dims d, double oe, const double* __restrict__ V, size_t sv,
                                                     const double* __restrict__ Wk, size_t sw, double* __restrict__ KV, size_t sk) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.nx) return;
  const int nline = DIR == 1 ? d.ny : d.nz;
  const int mline = nline + 2 * d.ng;
  const long long ls = DIR == 1 ? d.sy : d.sz;
  const int c0 = blockIdx.z * SEG;                           // first zone of the segment (interior index)
  const int other = blockIdx.y + d.ng;
  const long long base = (DIR == 1 ? (long long)other * d.sz : (long long)other * d.sy) + (i + d.ng);
  const int g0 = c0 + d.ng - 2;                              // line index of node 0 of the window (zone c0 - 2)
  // element offset of window node n inside a field, clamped (a ragged tail never reads past the field), in 32-bit arithmetic (a field has fewer than 2^32
  // points: checked at launch): min, multiply-add and one IMAD.WIDE per access instead of a 64-bit multiply-add chain
  const unsigned off0 = (unsigned)(base + (long long)g0 * ls), ls32 = (unsigned)ls;
  const int nmax = mline - 1 - g0;
  auto node = [&](int n) { return off0 + (unsigned)min(n, nmax) * ls32; };
  const double h = DIR == 1 ? d.dy : d.dz, ih = 1.0 / h;
#pragma unroll 1
  for (int s = 0; s < 3; ++s) {
    const double* wk = Wk + (size_t)(M1W * s) * sw;
    // face m (m = 0..SEG) lies between window nodes m + 1 and m + 2
    double lam[SEG + 1], A[SEG + 1];
    {
      const double* wl = wk + (size_t)(6 * DIR + 5) * sw;
      const double* wkap = wk + (size_t)18 * sw;
      double lp = __ldg(wl + node(1)), kp = __ldg(wkap + node(1));
#pragma unroll
      for (int m = 0; m <= SEG; ++m) {
        const double ln = __ldg(wl + node(m + 2)), kn = __ldg(wkap + node(m + 2));
        lam[m] = tmax(lp, ln);
        const double kh = 0.5 * (kp + kn) * h;
        A[m] = kh > 0.05 ? tanh(1.0 / kh) : 1.0;
        lp = ln; kp = kn;
      }
    }
#pragma unroll 1
    for (int f = 0; f < 5; ++f) {
      const double* u = V + (size_t)(5 * s + f) * sv;
      const double* F = wk + (size_t)(6 * DIR + f) * sw;
      double* kv = KV + (size_t)(5 * s + f) * sk;
      double uw[SEG + 4], Fw[SEG + 2], kold[SEG];
#pragma unroll
      for (int n = 0; n < SEG + 4; ++n) uw[n] = __ldg(u + node(n));
#pragma unroll
      for (int n = 0; n < SEG + 2; ++n) Fw[n] = __ldg(F + node(n + 1));
#pragma unroll
      for (int z = 0; z < SEG; ++z) kold[z] = kv[node(z + 2)];   // unconditional (clamped offsets); zones that do not exist are not stored
      double prev = m1_face(uw[0], uw[1], uw[2], uw[3], Fw[0], Fw[1], lam[0], A[0], oe);
#pragma unroll
      for (int z = 0; z < SEG; ++z) {
        const double cur = m1_face(uw[z + 1], uw[z + 2], uw[z + 3], uw[z + 4], Fw[z + 1], Fw[z + 2], lam[z + 1], A[z + 1], oe);
        if (c0 + z < nline) kv[node(z + 2)] = kold[z] - (cur - prev) * ih;
        prev = cur;
      }
    }
  }
}

cudaError_t launch_m1_point(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, const double* V, size_t sv,
                            double* Wk, size_t sw, cudaStream_t s) {
  k_m1_point<<<(unsigned)((d.npts + 127) / 128), 128, 0, s>>>(d, par, U, su, P, sp, V, sv, Wk, sw);
  return cudaGetLastError();
}
cudaError_t launch_m1_div(const Dims& d, const Par& par, const double* U, size_t su, const double* V, size_t sv, const double* Wk, size_t sw,
                          double* KV, size_t sk, cudaStream_t s) {
  const double oe = par.m1_odd_even != 0 ? par.m1_oe_guard : -1.0;
  if ((unsigned long long)d.npts >= (1ull << 32)) return cudaErrorInvalidValue;   // k_m1_march keeps 32-bit element offsets inside a field
  k_m1_div<<<dim3((d.nx + 15) / 16, (d.ny + 3) / 4, (d.nz + 1) / 2), dim3(16, 4, 2), 0, s>>>(d, oe, U, su, V, sv, Wk, sw, KV, sk);
  constexpr int SEG = 6;
  k_m1_march<1, SEG><<<dim3((d.nx + 127) / 128, d.nz, (d.ny + SEG - 1) / SEG), 128, 0, s>>>(d, oe, V, sv, Wk, sw, KV, sk);
  k_m1_march<2, SEG><<<dim3((d.nx + 127) / 128, d.ny, (d.nz + SEG - 1) / SEG), 128, 0, s>>>(d, oe, V, sv, Wk, sw, KV, sk);
  return cudaGetLastError();
}
cudaError_t launch_m1_implicit(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* V, size_t sv,
                               double* R, size_t sr, double adt, uint8_t* flags, cudaStream_t s) {
  k_m1_implicit<<<(unsigned)((d.npts + 127) / 128), 128, 0, s>>>(d, par, U, su, P, sp, V, sv, R, sr, adt, flags);
  return cudaGetLastError();
}
cudaError_t launch_m1_backreact(const Dims& d, const Par& par, const double* R, size_t sr, double* K, size_t sk, cudaStream_t s) {
  dim3 grid((d.nx + 127) / 128, d.ny, d.nz);
  k_m1_backreact<<<grid, 128, 0, s>>>(d, par.m1_mb, R, sr, K, sk);
  return cudaGetLastError();
}

}  // namespace mhd

// ---------------------------------------------------------------------------------------------------------------
// a4 with M1 on (R6, second half): E, F_i, P_ij of the three species added to the matter sources of Eqs. (14), (16), (17),
// (19), which are linear in them. P_ij is read from the M1 work slot (written by k_m1_point for the same V).
namespace mhd {
__global__ void __launch_bounds__(128) k_m1_gravity(const __grid_constant__ Dims d, double G8, const double* __restrict__ U, size_t su,
                                                    const double* __restrict__ V, size_t sv, const double* __restrict__ Wk, size_t sw,
                                                    double* __restrict__ K, size_t sk) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.nx) return;
  const size_t pt = (size_t)(blockIdx.z + d.ng) * d.sz + (size_t)(blockIdx.y + d.ng) * d.sy + (i + d.ng);
  double g[6], gi[6];
#pragma unroll
  for (int a = 0; a < 6; ++a) g[a] = __ldg(U + (size_t)(GXX + a) * su + pt);
  const double chi = __ldg(U + (size_t)CHI * su + pt), al = __ldg(U + (size_t)ALPHA * su + pt);
  {
    const double idet = 1.0 / (g[0] * (g[3] * g[5] - g[4] * g[4]) - g[1] * (g[1] * g[5] - g[4] * g[2]) + g[2] * (g[1] * g[4] - g[3] * g[2]));
    gi[0] = (g[3] * g[5] - g[4] * g[4]) * idet; gi[1] = (g[2] * g[4] - g[1] * g[5]) * idet; gi[2] = (g[1] * g[4] - g[2] * g[3]) * idet;
    gi[3] = (g[0] * g[5] - g[2] * g[2]) * idet; gi[4] = (g[1] * g[2] - g[0] * g[4]) * idet; gi[5] = (g[0] * g[3] - g[1] * g[1]) * idet;
  }
  const double isg = chi * sqrt(chi);
  double E = 0.0, F[3] = {0.0, 0.0, 0.0}, Pl[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    E += __ldg(V + (size_t)(5 * s + 1) * sv + pt) * isg;
#pragma unroll
    for (int a = 0; a < 3; ++a) F[a] += __ldg(V + (size_t)(5 * s + 2 + a) * sv + pt) * isg;
#pragma unroll
    for (int a = 0; a < 6; ++a) Pl[a] += __ldg(Wk + (size_t)(M1W * s + 19 + a) * sw + pt);
  }
  // gamma~^kl P_kl  (S = gamma^kl P_kl = chi times it)
  const double trt = gi[0] * Pl[0] + gi[3] * Pl[3] + gi[5] * Pl[5] + 2.0 * (gi[1] * Pl[1] + gi[2] * Pl[2] + gi[4] * Pl[4]);
  K[(size_t)KHAT * sk + pt] += al * 0.5 * G8 * (E + chi * trt);
  K[(size_t)THETA * sk + pt] -= al * G8 * E;
#pragma unroll
  for (int a = 0; a < 6; ++a) K[(size_t)(AXX + a) * sk + pt] -= al * G8 * chi * (Pl[a] - g[a] * trt * (1.0 / 3.0));
#pragma unroll
  for (int a = 0; a < 3; ++a)
    K[(size_t)(GAMX + a) * sk + pt] -= 2.0 * al * G8 * (gi[sy(a, 0)] * F[0] + gi[sy(a, 1)] * F[1] + gi[sy(a, 2)] * F[2]);
}

cudaError_t launch_m1_gravity(const Dims& d, const Par& par, const double* U, size_t su, const double* V, size_t sv, const double* Wk, size_t sw,
                              double* K, size_t sk, cudaStream_t s) {
  const double G8 = 8.0 * 3.14159265358979323846 * par.grav_G;
  if (G8 == 0.0) return cudaSuccess;
  dim3 grid((d.nx + 127) / 128, d.ny, d.nz);
  k_m1_gravity<<<grid, 128, 0, s>>>(d, G8, U, su, V, sv, Wk, sw, K, sk);
  return cudaGetLastError();
}
}  // namespace mhd
