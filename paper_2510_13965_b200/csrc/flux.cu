// a6-a7: GRMHD flux divergence, Eq. (32) flux brackets (l.256-260) discretised with the conservative
// finite-difference HRSC scheme of Sec. III C: Lax-Friedrichs flux splitting (Eq. 65) with the speed bound of
// App. B (Eqs. B1-B3, reading R12), MP5 reconstruction (Eqs. 67-76) and the flux sum (Eq. 69); Eq. (64).
//
// One kernel per direction, one thread per NODE of a line segment (interior nodes + 3 halo nodes per side):
//   phase 1  every node evaluates its pointwise flux F^d(U,P) (10 fields), keeps its conserved state U and its
//            speed bound s, and parks them in shared memory (computed once per node and direction);
//   phase 2  every interface i+1/2 takes lambda = max s over its six stencil nodes, splits F+- = (F +- lambda U)/2,
//            reconstructs F^L = MP5(F+ at i-2..i+2), F^R = MP5(F- at i+3..i-1) and sums them;
//   phase 3  every interior node subtracts (F^_{i+1/2} - F^_{i-1/2}) / h from K (the sources were written by ccz4.cu).
// Warps always run along x, so global loads/stores coalesce in all three directions; along y and z the line
// neighbours sit 32 threads apart in shared memory (conflict-free, no shuffles needed).
#include "mhd_internal.cuh"

namespace mhd {

namespace {

constexpr int NQ = 21;   // 10 fluxes + 10 conserved + 1 speed per node

__device__ __forceinline__ double minmod2(double a, double b) {
  const double m = fmin(fabs(a), fabs(b));
  return (a > 0.0 && b > 0.0) ? m : ((a < 0.0 && b < 0.0) ? -m : 0.0);
}
__device__ __forceinline__ double minmod4(double a, double b, double c, double d) {
  const double m = fmin(fmin(fabs(a), fabs(b)), fmin(fabs(c), fabs(d)));
  const bool pos = a > 0.0 && b > 0.0 && c > 0.0 && d > 0.0;
  const bool neg = a < 0.0 && b < 0.0 && c < 0.0 && d < 0.0;
  return pos ? m : (neg ? -m : 0.0);
}
// R_MP5(F_{i-2},...,F_{i+2}), Eqs. (70)-(76)
__device__ __forceinline__ double mp5(double fm2, double fm1, double f0, double fp1, double fp2, double alpha) {
  const double fhi = (2.0 * fm2 - 13.0 * fm1 + 47.0 * f0 + 27.0 * fp1 - 3.0 * fp2) * (1.0 / 60.0);
  const double dmh = f0 - fm1, dph = fp1 - f0;
  const double fmp = f0 + minmod2(dph, alpha * dmh);
  if ((fhi - f0) * (fhi - fmp) < 0.0) return fhi;
  const double dm1 = fm2 - 2.0 * fm1 + f0, d0 = fm1 - 2.0 * f0 + fp1, dp1 = f0 - 2.0 * fp1 + fp2;
  const double d4p = minmod4(4.0 * d0 - dp1, 4.0 * dp1 - d0, d0, dp1);
  const double d4m = minmod4(4.0 * dm1 - d0, 4.0 * d0 - dm1, dm1, d0);
  const double ful = f0 + alpha * dmh;
  const double fmd = 0.5 * (f0 + fp1) - 0.5 * d4p;
  const double flc = f0 + 0.5 * dmh + (4.0 / 3.0) * d4m;
  const double fmin_ = fmax(fmin(fmin(f0, fp1), fmd), fmin(fmin(f0, ful), flc));
  const double fmax_ = fmin(fmax(fmax(f0, fp1), fmd), fmax(fmax(f0, ful), flc));
  return fmin_ + minmod2(fhi - fmin_, fmax_ - fmin_);      // Median(fmin, fhi, fmax)
}

// pointwise flux brackets of Eq. (32) in direction DIR and the speed bound (App. B)
template <int DIR>
__device__ __forceinline__ void point_flux(const Par& par, const double* __restrict__ U, size_t su, const double* __restrict__ P, size_t sp,
                                           size_t pt, double F[10], double uc[10], double& smax) {
  auto u = [&](int f) { return __ldg(U + (size_t)f * su + pt); };
  auto pr = [&](int f) { return __ldg(P + (size_t)f * sp + pt); };
  const double gxx = u(GXX), gxy = u(GXY), gxz = u(GXZ), gyy = u(GYY), gyz = u(GYZ), gzz = u(GZZ);
  const double chi = u(CHI), al = u(ALPHA);
  const double be[3] = {u(BETAX), u(BETAY), u(BETAZ)};
#pragma unroll
  for (int a = 0; a < 10; ++a) uc[a] = u(DBAR + a);
  const double rho = pr(RHO), eps = pr(EPS), p = pr(PRESS), W = pr(WLOR), cs2 = pr(CS2);
  const double v[3] = {pr(VX), pr(VY), pr(VZ)};
  // row DIR of the inverse conformal metric (only gamma~^{DIR j} is needed)
  const double idet = 1.0 / (gxx * (gyy * gzz - gyz * gyz) - gxy * (gxy * gzz - gyz * gxz) + gxz * (gxy * gyz - gyy * gxz));
  double gid[3];
  if (DIR == 0) { gid[0] = (gyy * gzz - gyz * gyz) * idet; gid[1] = (gxz * gyz - gxy * gzz) * idet; gid[2] = (gxy * gyz - gxz * gyy) * idet; }
  if (DIR == 1) { gid[0] = (gxz * gyz - gxy * gzz) * idet; gid[1] = (gxx * gzz - gxz * gxz) * idet; gid[2] = (gxy * gxz - gxx * gyz) * idet; }
  if (DIR == 2) { gid[0] = (gxy * gyz - gxz * gyy) * idet; gid[1] = (gxy * gxz - gxx * gyz) * idet; gid[2] = (gxx * gyy - gxy * gxy) * idet; }
  const double ichi = 1.0 / chi;
  const double isg = chi * sqrt(chi), sg = 1.0 / isg;   // 1/sqrt(gamma), sqrt(gamma)
  // covariant velocity and magnetic field (physical metric gamma_ij = gamma~_ij / chi)
  const double Bu[3] = {uc[6] * isg, uc[7] * isg, uc[8] * isg};
  const double vl[3] = {ichi * (gxx * v[0] + gxy * v[1] + gxz * v[2]), ichi * (gxy * v[0] + gyy * v[1] + gyz * v[2]), ichi * (gxz * v[0] + gyz * v[1] + gzz * v[2])};
  const double Bl[3] = {ichi * (gxx * Bu[0] + gxy * Bu[1] + gxz * Bu[2]), ichi * (gxy * Bu[0] + gyy * Bu[1] + gyz * Bu[2]), ichi * (gxz * Bu[0] + gyz * Bu[1] + gzz * Bu[2])};
  const double v2 = v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2];
  const double B2 = Bu[0] * Bl[0] + Bu[1] * Bl[1] + Bu[2] * Bl[2];
  const double Bv = Bu[0] * vl[0] + Bu[1] * vl[1] + Bu[2] * vl[2];
  const double iW2 = 1.0 / (W * W);
  const double Sl[3] = {uc[3] * isg, uc[4] * isg, uc[5] * isg};
  // mixed stress S_i^DIR = gamma^{DIR j} S_ij with S_ij of l.260; gamma^{DIR j} gamma_ij = delta^DIR_i
  const double vd = v[DIR];                                                     // gamma^{dj} v_j = v^d
  const double Bd = Bu[DIR];
  const double Sd = chi * (gid[0] * Sl[0] + gid[1] * Sl[1] + gid[2] * Sl[2]);   // S^d
  const double ptot = p + 0.5 * (iW2 * B2 + Bv * Bv);                           // coefficient of gamma_ij in S_ij
  const double vk = al * vd - be[DIR];
  F[0] = vk * uc[0];
  F[1] = vk * uc[1];
  F[2] = -be[DIR] * uc[2] + al * (sg * Sd - uc[0] * vd);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const double Sid = 0.5 * (vl[i] * Sd + vd * Sl[i]) + (i == DIR ? ptot : 0.0) - iW2 * Bl[i] * Bd - 0.5 * Bv * (Bl[i] * vd + Bd * vl[i]);
    F[3 + i] = -be[DIR] * uc[3 + i] + al * sg * Sid;
    F[6 + i] = uc[6 + i] * vk - uc[6 + DIR] * (al * v[i] - be[i]) + al * chi * gid[i] * uc[9];
  }
  F[9] = -be[DIR] * uc[9] + al * par.c_b * par.c_b * uc[6 + DIR];
  // speed bound, Eqs. (B1)-(B3)
  const double h = rho * (1.0 + eps) + p;
  const double b2 = B2 * iW2 + Bv * Bv;
  const double ca2 = b2 / (h + b2);
  const double a2 = cs2 + ca2 - cs2 * ca2;
  const double gdd = chi * gid[DIR];
  const double disc = a2 * (1.0 - v2) * ((1.0 - v2 * a2) * gdd - (1.0 - a2) * vd * vd);
  const double root = sqrt(fmax(disc, 0.0));
  const double pre = al / (1.0 - v2 * a2);
  const double lp = -be[DIR] + pre * ((1.0 - a2) * vd + root);
  const double lm = -be[DIR] + pre * ((1.0 - a2) * vd - root);
  smax = fmax(fmax(fabs(lp), fabs(lm)), fabs(be[DIR]) + al * par.c_b * sqrt(gdd));
}

// NL nodes along the line per block; LS = distance in threads (and shared-memory slots) between line neighbours
template <int DIR, int NL, int NT>
__global__ void __launch_bounds__(NT) k_rhs_flux(const __grid_constant__ Dims d, const __grid_constant__ Par par,
                                                const double* __restrict__ U, size_t su, const double* __restrict__ P, size_t sp,
                                                double* __restrict__ K, size_t sk) {
  extern __shared__ double sh[];           // [NQ][NT]
  constexpr int TL = NL - 6;               // interior nodes per tile
  constexpr int LS = DIR == 0 ? 1 : NT / NL;
  const int tid = threadIdx.x;
  const int lpos = DIR == 0 ? tid % NL : tid / LS;      // position along the line
  const int lane = DIR == 0 ? tid / NL : tid % LS;      // which line of the block
  int ijk[3];
  bool valid;
  if (DIR == 0) {
    ijk[0] = d.ng - 3 + blockIdx.x * TL + lpos;
    ijk[1] = d.ng + blockIdx.y * (NT / NL) + lane;
    ijk[2] = d.ng + blockIdx.z;
    valid = ijk[0] < d.mx - (d.ng - 3) && ijk[1] < d.ng + d.ny;
  } else if (DIR == 1) {
    ijk[0] = d.ng + blockIdx.x * LS + lane;
    ijk[1] = d.ng - 3 + blockIdx.y * TL + lpos;
    ijk[2] = d.ng + blockIdx.z;
    valid = ijk[0] < d.ng + d.nx && ijk[1] < d.my - (d.ng - 3);
  } else {
    ijk[0] = d.ng + blockIdx.x * LS + lane;
    ijk[1] = d.ng + blockIdx.y;
    ijk[2] = d.ng - 3 + blockIdx.z * TL + lpos;
    valid = ijk[0] < d.ng + d.nx && ijk[2] < d.mz - (d.ng - 3);
  }
  const size_t pt = (size_t)ijk[2] * d.sz + (size_t)ijk[1] * d.sy + ijk[0];
  // ---- phase 1
  if (valid) {
    double F[10], uc[10], s;
    point_flux<DIR>(par, U, su, P, sp, pt, F, uc, s);
#pragma unroll
    for (int a = 0; a < 10; ++a) { sh[a * NT + tid] = F[a]; sh[(10 + a) * NT + tid] = uc[a]; }
    sh[20 * NT + tid] = s;
  }
  __syncthreads();
  // ---- phase 2: interface between lpos and lpos+1
  double Fh[10];
  const bool has_if = lpos >= 2 && lpos <= NL - 4;
  if (has_if) {
    double lam = 0.0;
#pragma unroll
    for (int m = -2; m <= 3; ++m) lam = fmax(lam, sh[20 * NT + tid + m * LS]);
#pragma unroll
    for (int a = 0; a < 10; ++a) {
      double fp[6], fm[6];
#pragma unroll
      for (int m = 0; m < 6; ++m) {
        const double f = sh[a * NT + tid + (m - 2) * LS], uu = sh[(10 + a) * NT + tid + (m - 2) * LS];
        fp[m] = 0.5 * (f + lam * uu);                                            // Eq. (65)
        fm[m] = 0.5 * (f - lam * uu);
      }
      Fh[a] = mp5(fp[0], fp[1], fp[2], fp[3], fp[4], par.mp5_alpha)              // Eq. (67)
              + mp5(fm[5], fm[4], fm[3], fm[2], fm[1], par.mp5_alpha);           // Eqs. (68), (69)
    }
  }
  __syncthreads();
  if (has_if) {
#pragma unroll
    for (int a = 0; a < 10; ++a) sh[a * NT + tid] = Fh[a];                        // F^_{lpos+1/2}
  }
  __syncthreads();
  // ---- phase 3: interior nodes of this tile
  const int gl = DIR == 0 ? ijk[0] : (DIR == 1 ? ijk[1] : ijk[2]);
  const int nd = DIR == 0 ? d.nx : (DIR == 1 ? d.ny : d.nz);
  if (valid && lpos >= 3 && lpos <= NL - 4 && gl < d.ng + nd) {
    const double ih = 1.0 / (DIR == 0 ? d.dx : (DIR == 1 ? d.dy : d.dz));
#pragma unroll
    for (int a = 0; a < 10; ++a) {
      double* kp = K + (size_t)(DBAR + a) * sk + pt;
      *kp -= (sh[a * NT + tid] - sh[a * NT + tid - LS]) * ih;                      // Eq. (64)
    }
  }
}

template <int DIR, int NL, int NT>
cudaError_t launch_dir(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* K, size_t sk, cudaStream_t s) {
  constexpr int TL = NL - 6;
  constexpr size_t smem = (size_t)NQ * NT * sizeof(double);
  auto kern = k_rhs_flux<DIR, NL, NT>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid;
  if (DIR == 0) grid = dim3((d.nx + TL - 1) / TL, (d.ny + NT / NL - 1) / (NT / NL), d.nz);
  if (DIR == 1) grid = dim3((d.nx + NT / NL - 1) / (NT / NL), (d.ny + TL - 1) / TL, d.nz);
  if (DIR == 2) grid = dim3((d.nx + NT / NL - 1) / (NT / NL), d.ny, (d.nz + TL - 1) / TL);
  kern<<<grid, NT, smem, s>>>(d, par, U, su, P, sp, K, sk);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_rhs_flux(int dir, const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* K, size_t sk, cudaStream_t s) {
  if (dir == 0) return launch_dir<0, 64, 256>(d, par, U, su, P, sp, K, sk, s);
  if (dir == 1) return launch_dir<1, 16, 512>(d, par, U, su, P, sp, K, sk, s);
  return launch_dir<2, 16, 512>(d, par, U, su, P, sp, K, sk, s);
}

}  // namespace mhd
