// a6-a7: GRMHD flux divergence, Eq. (32) flux brackets (l.256-260) discretised with the conservative
// finite-difference HRSC scheme of Sec. III C: Lax-Friedrichs flux splitting (Eq. 65) with the speed bound of
// App. B (Eqs. B1-B3, reading R12), MP5 reconstruction (Eqs. 67-76) and the flux sum (Eq. 69); Eq. (64).
//
// Two steps:
//   k_point_flux   every grid point (ghosts included) evaluates ONCE the flux brackets F^x, F^y, F^z of the 10 fluid
//                  fields and the three speed bounds s^x, s^y, s^z (the inverse metric, covariant v and B, b^2 ...
//                  are shared between the directions) and writes them to the 33-field work slot
//                  (field 11 d + a: a = 0..9 flux of field a in direction d, a = 10 speed).
//   k_recon<DIR>   streaming 1-D kernels: per interface lambda = max s over its six stencil nodes, F+- = F +- lambda U
//                  (the factor 1/2 of Eq. 65 is applied after the reconstruction: R_MP5 is homogeneous of degree one
//                  and scaling by 1/2 is exact), F^L = MP5(F+ at i-2..i+2), F^R = MP5(F- at i+3..i-1), Eq. (69),
//                  and K -= (F^_{i+1/2} - F^_{i-1/2}) / h (the sources were written to K by ccz4.cu).
//                  y and z: one thread marches along a segment of SEG zones with a 6-node register window per field,
//                  warps run along x (coalesced), every node value is loaded once per segment.
//                  x: one thread per interface, six L1-resident loads per array, the left neighbour's F^ comes by
//                  warp shuffle.
// MP5: the limiter of Eqs. (73)-(76) is needed only where the test of Eq. (72) fails; the branch is taken per warp
// (__any_sync), so smooth regions run the 5-point formula of Eq. (70) alone. Sign / magnitude selections of
// minmod are done on the integer pipe (bit patterns of non-negative doubles order like integers), which keeps
// the FP64 pipe for arithmetic.
#include <stdlib.h>
#include "mhd_internal.cuh"

namespace mhd {

namespace {

constexpr long long SIGN = (long long)0x8000000000000000ULL;

__device__ __forceinline__ long long bits(double a) { return __double_as_longlong(a); }
__device__ __forceinline__ double dbl(long long a) { return __longlong_as_double(a); }
__device__ __forceinline__ double dmin(double a, double b) { return b < a ? b : a; }
__device__ __forceinline__ double dmax(double a, double b) { return a < b ? b : a; }
// max of two non-negative doubles on the integer pipe
__device__ __forceinline__ double pmax(double a, double b) { return dbl(max(bits(a), bits(b))); }

// minmod of two arguments: common sign x smallest magnitude, else 0 (R14)
__device__ __forceinline__ double minmod2(double a, double b) {
  const long long ia = bits(a), ib = bits(b);
  const long long m = min(ia & ~SIGN, ib & ~SIGN);
  return ((ia ^ ib) < 0) ? 0.0 : dbl(m | (ia & SIGN));
}
__device__ __forceinline__ double minmod4(double a, double b, double c, double d) {
  const long long ia = bits(a), ib = bits(b), ic = bits(c), id = bits(d);
  const long long m = min(min(ia & ~SIGN, ib & ~SIGN), min(ic & ~SIGN, id & ~SIGN));
  const bool neg = (ia & ib & ic & id) < 0, pos = (ia | ib | ic | id) >= 0;
  return (neg || pos) ? dbl(m | (ia & SIGN)) : 0.0;
}

// Eq. (70) and the test of Eq. (72). The test is a shortcut (DESIGN.md note N4): whenever f^hi lies between F_i and
// f^MP = F_i + minmod(dph, alpha dmh) the limiter of Eqs. (73)-(76) returns it unchanged. With t = f^hi - F_i that is
// "t between 0 and dph, and between 0 and alpha dmh": two products, no minmod. The closed interval (<=) is used: at
// its end points (t = 0: constant data, e.g. atmosphere; t = dph; t = alpha dmh) the limiter is still the identity.
__device__ __forceinline__ double mp5_hi(double fm2, double fm1, double f0, double fp1, double fp2, double alpha, bool& need) {
  const double fhi = (2.0 * fm2 - 13.0 * fm1 + 47.0 * f0 + 27.0 * fp1 - 3.0 * fp2) * (1.0 / 60.0);   // Eq. (70)
  const double t = fhi - f0;
  need = !((t * (t - (fp1 - f0)) <= 0.0) && (t * (t - alpha * (f0 - fm1)) <= 0.0));                  // Eqs. (71)-(72)
  return fhi;
}

// Median(f^hi, f^min, f^max) - f^hi, Eqs. (73)-(76): the correction the limiter applies to Eq. (70)
__device__ __forceinline__ double mp5_correction(double fm2, double fm1, double f0, double fp1, double fp2, double alpha) {
  const double fhi = (2.0 * fm2 - 13.0 * fm1 + 47.0 * f0 + 27.0 * fp1 - 3.0 * fp2) * (1.0 / 60.0);
  const double dmh = f0 - fm1;
  const double dm1 = fm2 - 2.0 * fm1 + f0, d0 = fm1 - 2.0 * f0 + fp1, dp1 = f0 - 2.0 * fp1 + fp2;
  const double d4p = minmod4(4.0 * d0 - dp1, 4.0 * dp1 - d0, d0, dp1);                               // Eq. (76)
  const double d4m = minmod4(4.0 * dm1 - d0, 4.0 * d0 - dm1, dm1, d0);
  const double ful = f0 + alpha * dmh;                                                               // Eq. (73)
  const double fmd = 0.5 * (f0 + fp1) - 0.5 * d4p;                                                   // Eq. (74)
  const double flc = f0 + 0.5 * dmh + (4.0 / 3.0) * d4m;                                             // Eq. (75)
  const double lo = dmax(dmin(dmin(f0, fp1), fmd), dmin(dmin(f0, ful), flc));
  const double hi = dmin(dmax(dmax(f0, fp1), fmd), dmax(dmax(f0, ful), flc));
  return (lo - fhi) + minmod2(fhi - lo, hi - lo);                                                    // Median(lo, fhi, hi) - fhi
}

// ---------------------------------------------------------------------------------------------------------------
// Warp-divergence control for the limiter. Only a fraction of the reconstructions fail the test of Eq. (72)
// (near extrema, discontinuities), but in a 32-wide warp almost every warp holds one, so a per-lane branch would
// run the limiter for everybody. Instead each lane pushes the five stencil values of its failing reconstructions
// on a per-warp stack in shared memory; whenever 32 are pending the warp pops them and evaluates the limiter
// densely, one entry per lane, and posts the correction to the owner's slot. The owner adds it afterwards.
// ---------------------------------------------------------------------------------------------------------------
constexpr int QCAP = 96;                 // 32 pending + up to 64 pushed between two flushes
constexpr unsigned FULL = 0xffffffffu;

struct LimQueue {
  double* v;       // [5][QCAP] stencil values F_{i-2}..F_{i+2} of the pending reconstructions
  int* tag;        // [QCAP]    owner lane | slot << 5
  double* corr;    // [NSLOT][32] corrections by slot and owner lane
  int count;       // pending entries (warp-uniform)
};

__device__ __forceinline__ void q_push(LimQueue& q, bool need, double fm2, double fm1, double f0, double fp1, double fp2, int slot, int lane) {
  const unsigned b = __ballot_sync(FULL, need);
  if (need) {
    const int pos = q.count + __popc(b & ((1u << lane) - 1u));
    q.v[pos] = fm2; q.v[QCAP + pos] = fm1; q.v[2 * QCAP + pos] = f0; q.v[3 * QCAP + pos] = fp1; q.v[4 * QCAP + pos] = fp2;
    q.tag[pos] = lane | (slot << 5);
  }
  q.count += __popc(b);
}
// evaluate entries [first, first + n), n <= 32, one per lane
__device__ __noinline__ void q_process(const double* v, const int* tag, double* corr, int first, int n, int lane, double alpha) {
  __syncwarp();
  if (lane < n) {
    const int e = first + lane;
    const int tg = tag[e];
    corr[(tg >> 5) * 32 + (tg & 31)] = mp5_correction(v[e], v[QCAP + e], v[2 * QCAP + e], v[3 * QCAP + e], v[4 * QCAP + e], alpha);
  }
  __syncwarp();
}
__device__ __forceinline__ void q_flush(LimQueue& q, int lane, double alpha) {
  while (q.count >= 32) { q.count -= 32; q_process(q.v, q.tag, q.corr, q.count, 32, lane, alpha); }
}
__device__ __forceinline__ void q_drain(LimQueue& q, int lane, double alpha) {
  q_flush(q, lane, alpha);
  if (q.count > 0) { q_process(q.v, q.tag, q.corr, 0, q.count, lane, alpha); q.count = 0; }
}

// WENO5, the second reconstruction named at PAPER.md:486-488 (Jiang & Shu, ref. [63]): candidate values, smoothness indicators,
// linear weights (1/10, 6/10, 3/10), exponent 2, epsilon = weno_eps. One division per reconstruction; no branches, so no queue.
__device__ __forceinline__ double weno5(double fm2, double fm1, double f0, double fp1, double fp2, double eps) {
  const double q0 = (2.0 * fm2 - 7.0 * fm1 + 11.0 * f0) * (1.0 / 6.0);
  const double q1 = (-fm1 + 5.0 * f0 + 2.0 * fp1) * (1.0 / 6.0);
  const double q2 = (2.0 * f0 + 5.0 * fp1 - fp2) * (1.0 / 6.0);
  const double c0 = fm2 - 2.0 * fm1 + f0, e0 = fm2 - 4.0 * fm1 + 3.0 * f0;
  const double c1 = fm1 - 2.0 * f0 + fp1, e1 = fm1 - fp1;
  const double c2 = f0 - 2.0 * fp1 + fp2, e2 = 3.0 * f0 - 4.0 * fp1 + fp2;
  const double b0 = eps + ((13.0 / 12.0) * c0 * c0 + 0.25 * e0 * e0);
  const double b1 = eps + ((13.0 / 12.0) * c1 * c1 + 0.25 * e1 * e1);
  const double b2 = eps + ((13.0 / 12.0) * c2 * c2 + 0.25 * e2 * e2);
  // a_k = d_k / b_k^2 over the common denominator (b0 b1 b2)^2: w_k = d_k (b_l b_m)^2 / sum
  const double n0 = 0.1 * (b1 * b2) * (b1 * b2), n1 = 0.6 * (b0 * b2) * (b0 * b2), n2 = 0.3 * (b0 * b1) * (b0 * b1);
  return (n0 * q0 + n1 * q1 + n2 * q2) / (n0 + n1 + n2);
}

// Eqs. (65), (67)-(69) for one interface and one field from the six stencil nodes i-2..i+3 (index 0..5): returns
// f^hi_L + f^hi_R (twice the unlimited F^) and queues the reconstructions that need the limiter (slots 2s, 2s+1).
// WENO: `alpha` carries weno_eps; the weights are not homogeneous in F, so the 1/2 of Eq. (65) is applied before the reconstruction
// and the sum is doubled again (exact) to keep the caller's 1/(2h).
template <bool WENO>
__device__ __forceinline__ double flux_hat2(LimQueue& q, const double f[6], const double u[6], double lam, double alpha, bool active,
                                            int s, int lane, unsigned& mask) {
  double p[5], m[5];
  if (WENO) {
#pragma unroll
    for (int n = 0; n < 5; ++n) { p[n] = 0.5 * fma(lam, u[n], f[n]); m[n] = 0.5 * fma(-lam, u[n + 1], f[n + 1]); }
    return 2.0 * (weno5(p[0], p[1], p[2], p[3], p[4], alpha) + weno5(m[4], m[3], m[2], m[1], m[0], alpha));
  }
#pragma unroll
  for (int n = 0; n < 5; ++n) { p[n] = fma(lam, u[n], f[n]); m[n] = fma(-lam, u[n + 1], f[n + 1]); }
  bool nl, nr;
  const double fl = mp5_hi(p[0], p[1], p[2], p[3], p[4], alpha, nl);
  const double fr = mp5_hi(m[4], m[3], m[2], m[1], m[0], alpha, nr);
  nl = nl && active; nr = nr && active;
  q_push(q, nl, p[0], p[1], p[2], p[3], p[4], 2 * s, lane);
  q_push(q, nr, m[4], m[3], m[2], m[1], m[0], 2 * s + 1, lane);
  mask |= ((unsigned)nl << (2 * s)) | ((unsigned)nr << (2 * s + 1));
  return fl + fr;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
// Pointwise flux brackets of Eq. (32) in all three directions and the speed bounds of App. B (Eqs. B1-B3, R12)
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_point_flux(const __grid_constant__ Dims d, const __grid_constant__ Par par,
                                                    const double* __restrict__ U, size_t su, const double* __restrict__ P, size_t sp,
                                                    double* __restrict__ Wk, size_t sw) {
  const long long pt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (pt >= d.npts) return;
  auto u = [&](int f) { return __ldg(U + (size_t)f * su + pt); };
  auto pr = [&](int f) { return __ldg(P + (size_t)f * sp + pt); };
  const double gxx = u(GXX), gxy = u(GXY), gxz = u(GXZ), gyy = u(GYY), gyz = u(GYZ), gzz = u(GZZ);
  const double chi = u(CHI), al = u(ALPHA);
  const double be[3] = {u(BETAX), u(BETAY), u(BETAZ)};
  double uc[10];
#pragma unroll
  for (int a = 0; a < 10; ++a) uc[a] = u(DBAR + a);
  const double rho = pr(RHO), eps = pr(EPS), p = pr(PRESS), W = pr(WLOR), cs2 = pr(CS2);
  const double v[3] = {pr(VX), pr(VY), pr(VZ)};
  const double idet = 1.0 / (gxx * (gyy * gzz - gyz * gyz) - gxy * (gxy * gzz - gyz * gxz) + gxz * (gxy * gyz - gyy * gxz));
  double gi[3][3];
  gi[0][0] = (gyy * gzz - gyz * gyz) * idet;
  gi[0][1] = gi[1][0] = (gxz * gyz - gxy * gzz) * idet;
  gi[0][2] = gi[2][0] = (gxy * gyz - gxz * gyy) * idet;
  gi[1][1] = (gxx * gzz - gxz * gxz) * idet;
  gi[1][2] = gi[2][1] = (gxy * gxz - gxx * gyz) * idet;
  gi[2][2] = (gxx * gyy - gxy * gxy) * idet;
  const double ichi = 1.0 / chi;
  const double isg = chi * sqrt(chi), sg = 1.0 / isg;   // 1/sqrt(gamma), sqrt(gamma)
  const double Bu[3] = {uc[6] * isg, uc[7] * isg, uc[8] * isg};
  const double vl[3] = {ichi * (gxx * v[0] + gxy * v[1] + gxz * v[2]), ichi * (gxy * v[0] + gyy * v[1] + gyz * v[2]), ichi * (gxz * v[0] + gyz * v[1] + gzz * v[2])};
  const double Bl[3] = {ichi * (gxx * Bu[0] + gxy * Bu[1] + gxz * Bu[2]), ichi * (gxy * Bu[0] + gyy * Bu[1] + gyz * Bu[2]), ichi * (gxz * Bu[0] + gyz * Bu[1] + gzz * Bu[2])};
  const double v2 = v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2];
  const double B2 = Bu[0] * Bl[0] + Bu[1] * Bl[1] + Bu[2] * Bl[2];
  const double Bv = Bu[0] * vl[0] + Bu[1] * vl[1] + Bu[2] * vl[2];
  const double iW2 = 1.0 / (W * W);
  const double Sl[3] = {uc[3] * isg, uc[4] * isg, uc[5] * isg};
  const double ptot = p + 0.5 * (iW2 * B2 + Bv * Bv);     // coefficient of gamma_ij in S_ij (l.260)
  const double h = rho * (1.0 + eps) + p;                 // enthalpy density (l.232)
  const double b2 = B2 * iW2 + Bv * Bv;                   // (B3)
  const double ca2 = b2 / (h + b2);
  const double a2 = cs2 + ca2 - cs2 * ca2;                // (B2)
  const double pre = al / (1.0 - v2 * a2);
  const double cb2 = par.c_b * par.c_b;
#pragma unroll
  for (int dir = 0; dir < 3; ++dir) {
    const double vd = v[dir], Bd = Bu[dir];
    const double Sd = chi * (gi[dir][0] * Sl[0] + gi[dir][1] * Sl[1] + gi[dir][2] * Sl[2]);   // S^d
    const double vk = al * vd - be[dir];
    double* out = Wk + (size_t)(11 * dir) * sw + pt;
    out[0] = vk * uc[0];
    out[sw] = vk * uc[1];
    out[2 * sw] = -be[dir] * uc[2] + al * (sg * Sd - uc[0] * vd);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      // mixed stress S_i^d = gamma^{dj} S_ij with S_ij of l.260 (gamma^{dj} gamma_ij = delta^d_i, gamma^{dj} v_j = v^d)
      const double Sid = 0.5 * (vl[i] * Sd + vd * Sl[i]) + (i == dir ? ptot : 0.0) - iW2 * Bl[i] * Bd - 0.5 * Bv * (Bl[i] * vd + Bd * vl[i]);
      out[(3 + i) * sw] = -be[dir] * uc[3 + i] + al * sg * Sid;
      out[(6 + i) * sw] = uc[6 + i] * vk - uc[6 + dir] * (al * v[i] - be[i]) + al * chi * gi[dir][i] * uc[9];
    }
    out[9 * sw] = -be[dir] * uc[9] + al * cb2 * uc[6 + dir];
    const double gdd = chi * gi[dir][dir];
    const double disc = a2 * (1.0 - v2) * ((1.0 - v2 * a2) * gdd - (1.0 - a2) * vd * vd);
    const double root = sqrt(fmax(disc, 0.0));
    const double lp = -be[dir] + pre * ((1.0 - a2) * vd + root);                               // (B1)
    const double lm = -be[dir] + pre * ((1.0 - a2) * vd - root);
    out[10 * sw] = fmax(fmax(fabs(lp), fabs(lm)), fabs(be[dir]) + al * par.c_b * sqrt(gdd));
  }
}

cudaError_t launch_point_flux(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* Wk, size_t sw, cudaStream_t s) {
  k_point_flux<<<(unsigned)((d.npts + 127) / 128), 128, 0, s>>>(d, par, U, su, P, sp, Wk, sw);
  return cudaGetLastError();
}

namespace {

// ---------------------------------------------------------------------------------------------------------------
// y / z: marching reconstruction. Thread = (x column, segment of SEG zones along the line). blockIdx.y = the third axis.
// All 32 lanes of a warp stay alive (the limiter queue is warp-cooperative): columns past nx are clamped and masked.
// ---------------------------------------------------------------------------------------------------------------
constexpr int RW = 4;    // warps per CTA of the reconstruction kernels
constexpr int RXROWS = 4;   // rows a warp of k_recon_x takes in turn

template <int DIR, int SEG, bool FUSED, bool WENO>
__global__ void __launch_bounds__(32 * RW, 4) k_recon_march(const __grid_constant__ Dims d, double alpha, const double* __restrict__ U, size_t su,
                                                            const double* __restrict__ Wk, size_t sw, double* __restrict__ K, size_t sk,
                                                            const __grid_constant__ Fuse fz) {
  __shared__ double q_v[RW][5 * QCAP];
  __shared__ int q_tag[RW][QCAP];
  __shared__ double q_corr[RW][2 * (SEG + 1) * 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  LimQueue q = {q_v[warp], q_tag[warp], q_corr[warp], 0};
  const int ii = blockIdx.x * blockDim.x + threadIdx.x;
  const bool active = ii < d.nx;
  const int i = min(ii, d.nx - 1);
  const int nline = DIR == 1 ? d.ny : d.nz;
  const int mline = nline + 2 * d.ng;
  const long long ls = DIR == 1 ? d.sy : d.sz;               // stride along the line
  const int c0 = blockIdx.z * SEG;                           // first zone of the segment (interior index)
  // base = node (c0 - 3) of the line, i.e. global line index c0 + ng - 3
  const int other = blockIdx.y + d.ng;
  const long long base = (DIR == 1 ? (long long)other * d.sz : (long long)other * d.sy) + (i + d.ng);
  const int g0 = c0 + d.ng - 3;
  // element offset of node n of the segment inside a field, clamped (the ragged tail never reads past the field), in 32-bit arithmetic (a field has fewer
  // than 2^32 points: checked at launch): min, multiply-add, IMAD.WIDE per access instead of a 64-bit multiply-add chain
  const unsigned off0 = (unsigned)(base + (long long)g0 * ls), ls32 = (unsigned)ls;
  const int nmax = mline - 1 - g0;
  auto offn = [&](int n) { return off0 + (unsigned)min(n, nmax) * ls32; };
  // lambda of the SEG+1 interfaces: interface m lies between nodes m+2 and m+3 (relative to g0), stencil nodes m..m+5
  double lam[SEG + 1];
  {
    const double* s = Wk + (size_t)(11 * DIR + 10) * sw;
    double w[6];
#pragma unroll
    for (int n = 0; n < 5; ++n) w[n] = __ldg(s + offn(n));
#pragma unroll
    for (int m = 0; m <= SEG; ++m) {
      w[(m + 5) % 6] = __ldg(s + offn(m + 5));
      lam[m] = pmax(pmax(pmax(w[0], w[1]), pmax(w[2], w[3])), pmax(w[4], w[5]));
    }
  }
  const double hih = 0.5 / (DIR == 1 ? d.dy : d.dz);         // the 1/2 of Eq. (65) and 1/h of Eq. (64)
#pragma unroll 1
  for (int a = 0; a < 10; ++a) {
    const double* f = Wk + (size_t)(11 * DIR + a) * sw;
    const double* u = U + (size_t)(DBAR + a) * su;
    double* k = K + (size_t)(DBAR + a) * sk;
    // the whole column of the segment (SEG + 6 nodes) is loaded up front: the warp-synchronous limiter queue below
    // fences code motion, so loads issued inside the interface loop would each expose a full memory latency
    double fc[SEG + 6], uc[SEG + 6], acc[SEG + 1];
    unsigned mask = 0;
#pragma unroll
    for (int n = 0; n < SEG + 6; ++n) { fc[n] = __ldg(f + offn(n)); uc[n] = __ldg(u + offn(n)); }
    double kold[SEG];                                          // K is read-modify-write: fetched with the column, not after the arithmetic
#pragma unroll
    for (int m = 1; m <= SEG; ++m) kold[m - 1] = k[offn(m + 2)];   // unconditional: the offsets are clamped into the field, zones that do not exist are not stored
    double pre[SEG];                                           // U0 + earlier stages of the fused RK combine (z pass only), fetched with the rest
#pragma unroll
    for (int m = 1; m <= SEG; ++m) pre[m - 1] = (FUSED && active && c0 + m - 1 < nline) ? fused_fetch(fz, DBAR + a, (size_t)offn(m + 2)) : 0.0;
#pragma unroll
    for (int m = 0; m <= SEG; ++m) {
      acc[m] = flux_hat2<WENO>(q, fc + m, uc + m, lam[m], alpha, active, m, lane, mask);
      if (!WENO) q_flush(q, lane, alpha);
    }
    if (!WENO) q_drain(q, lane, alpha);
#pragma unroll
    for (int m = 0; m <= SEG; ++m) {
      if (mask & (1u << (2 * m))) acc[m] += q.corr[(2 * m) * 32 + lane];
      if (mask & (1u << (2 * m + 1))) acc[m] += q.corr[(2 * m + 1) * 32 + lane];
    }
#pragma unroll
    for (int m = 1; m <= SEG; ++m)
      if (active && c0 + m - 1 < nline) {
        const size_t pt = offn(m + 2);                                   // zone c0 + m - 1
        const double knew = kold[m - 1] - (acc[m] - acc[m - 1]) * hih;          // Eq. (64)
        if (FUSED) fused_store(fz, DBAR + a, pt, pre[m - 1], knew, k + pt); else k[pt] = knew;
      }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// x: one thread per interface; a warp covers 32 interfaces = 31 zones (lane 31 only supplies F^ to lane 30).
// ---------------------------------------------------------------------------------------------------------------
template <bool WENO>
__global__ void __launch_bounds__(32 * RW, 4) k_recon_x(const __grid_constant__ Dims d, double alpha, const double* __restrict__ U, size_t su,
                                                        const double* __restrict__ Wk, size_t sw, double* __restrict__ K, size_t sk) {
  __shared__ double q_v[RW][5 * QCAP];
  __shared__ int q_tag[RW][QCAP];
  __shared__ double q_corr[RW][20 * 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  LimQueue q = {q_v[warp], q_tag[warp], q_corr[warp], 0};
  const int z0 = blockIdx.x * 31;                            // first zone of this warp
  const int zone = z0 + lane;                                // lane l: interface zone-1/2 (left face of its zone)
  // a warp takes RXROWS consecutive rows (j), one after the other: while it works on one, the first lines of the next are pulled into L1, so that the round
  // trip of a row's first loads (lambda, K, field 0) is exposed once per RXROWS rows
#pragma unroll 1
  for (int r = 0; r < RXROWS; ++r) {
  const int row = (blockIdx.y * RW + warp) * RXROWS + r;     // j index (interior)
  if (row >= d.ny) return;                                   // whole warp leaves
  // left face of zone: between nodes zone-1 and zone -> stencil nodes zone-3 .. zone+2 ; global x index = zone + ng - 3 + n
  const long long base = (long long)(blockIdx.z + d.ng) * d.sz + (long long)(row + d.ng) * d.sy;
  // lanes past the last interface (zone > nx) are clamped as a whole, so that the six nodes of every lane are contiguous and inside the row (ng >= 3): a
  // load is [pointer + immediate], the pointer of a field one IMAD.WIDE from the 32-bit element offset of node 0 (a field has fewer than 2^32 points)
  const unsigned off0 = (unsigned)(base + (min(zone, d.nx) + d.ng - 3));
  auto node = [&](int n) { return (size_t)off0 + n; };
  const bool active = zone <= d.nx;                          // interfaces 0 .. nx
  if (r + 1 < RXROWS && row + 1 < d.ny) {
    const size_t nx2 = (size_t)off0 + (size_t)d.sy + 2;      // node 2 of the next row
    asm volatile("prefetch.global.L1 [%0];" ::"l"(Wk + (size_t)10 * sw + nx2));
    asm volatile("prefetch.global.L1 [%0];" ::"l"(Wk + nx2));
    asm volatile("prefetch.global.L1 [%0];" ::"l"(U + (size_t)DBAR * su + nx2));
#pragma unroll
    for (int a = 0; a < 10; ++a) asm volatile("prefetch.global.L1 [%0];" ::"l"(K + (size_t)(DBAR + a) * sk + nx2 + 1));
  }
  double lam;
  {
    const double* s = Wk + (size_t)10 * sw;
    lam = pmax(pmax(pmax(__ldg(s + node(0)), __ldg(s + node(1))), pmax(__ldg(s + node(2)), __ldg(s + node(3)))), pmax(__ldg(s + node(4)), __ldg(s + node(5))));
  }
  const double hih = 0.5 / d.dx;
  const bool store = lane < 31 && zone < d.nx;
  double acc[10], kold[10];
  unsigned mask = 0;
#pragma unroll
  for (int a = 0; a < 10; ++a) kold[a] = K[(size_t)(DBAR + a) * sk + off0 + 3];   // read-modify-write: fetched up front, unconditionally (the clamped node is inside the row)
  double fw[6], uw[6];
#pragma unroll
  for (int n = 0; n < 6; ++n) { fw[n] = __ldg(Wk + node(n)); uw[n] = __ldg(U + (size_t)DBAR * su + node(n)); }
#pragma unroll
  for (int a = 0; a < 10; ++a) {
    double fn[6], un[6];                                      // next field's stencil, in flight during this field's arithmetic
    if (a < 9) {
      const double* f = Wk + (size_t)(a + 1) * sw;
      const double* u = U + (size_t)(DBAR + a + 1) * su;
#pragma unroll
      for (int n = 0; n < 6; ++n) { fn[n] = __ldg(f + node(n)); un[n] = __ldg(u + node(n)); }
    }
    if (a < 8) {                                               // and the field after that is pulled into L1 (no registers to hold it)
      asm volatile("prefetch.global.L1 [%0];" ::"l"(Wk + (size_t)(a + 2) * sw + node(2)));
      asm volatile("prefetch.global.L1 [%0];" ::"l"(U + (size_t)(DBAR + a + 2) * su + node(2)));
    }
    acc[a] = flux_hat2<WENO>(q, fw, uw, lam, alpha, active, a, lane, mask);   // twice F^ at zone - 1/2
    if (!WENO) q_flush(q, lane, alpha);
    if (a < 9) {
#pragma unroll
      for (int n = 0; n < 6; ++n) { fw[n] = fn[n]; uw[n] = un[n]; }
    }
  }
  if (!WENO) q_drain(q, lane, alpha);
#pragma unroll
  for (int a = 0; a < 10; ++a) {
    double fl = acc[a];
    if (mask & (1u << (2 * a))) fl += q.corr[(2 * a) * 32 + lane];
    if (mask & (1u << (2 * a + 1))) fl += q.corr[(2 * a + 1) * 32 + lane];
    const double fr = __shfl_down_sync(FULL, fl, 1);           // F^ at zone + 1/2
    if (store) K[(size_t)(DBAR + a) * sk + off0 + 3] = kold[a] - (fr - fl) * hih;
  }
  }
}

}  // namespace

template <int SEG, bool WENO>
static void launch_march(int dir, const Dims& d, const Par& par, const double* U, size_t su, const double* Wk, size_t sw, double* K, size_t sk, const Fuse& fz, cudaStream_t s) {
  const double a = WENO ? par.weno_eps : par.mp5_alpha;
  if (dir == 1) {
    dim3 grid((d.nx + 32 * RW - 1) / (32 * RW), d.nz, (d.ny + SEG - 1) / SEG);
    k_recon_march<1, SEG, false, WENO><<<grid, 32 * RW, 0, s>>>(d, a, U, su, Wk, sw, K, sk, fz);
  } else {                                                                    // z is the last pass over the fluid K: the RK combine rides on it
    dim3 grid((d.nx + 32 * RW - 1) / (32 * RW), d.ny, (d.nz + SEG - 1) / SEG);
    if (fz.Uout) k_recon_march<2, SEG, true, WENO><<<grid, 32 * RW, 0, s>>>(d, a, U, su, Wk, sw, K, sk, fz);
    else k_recon_march<2, SEG, false, WENO><<<grid, 32 * RW, 0, s>>>(d, a, U, su, Wk, sw, K, sk, fz);
  }
}

cudaError_t launch_recon(int dir, const Dims& d, const Par& par, const double* U, size_t su, const double* Wk, size_t sw, double* K, size_t sk, const Fuse& fz, cudaStream_t s) {
  static int seg = 0;
  if (seg == 0) { const char* v = getenv("MHD_RECON_SEG"); seg = v ? atoi(v) : 6; }
  const bool weno = par.recon_kind == 1;
  if ((unsigned long long)d.npts >= (1ull << 32)) return cudaErrorInvalidValue;   // the kernels keep 32-bit element offsets inside a field
  if (dir == 0) {
    dim3 grid((d.nx + 30) / 31, (d.ny + RW * RXROWS - 1) / (RW * RXROWS), d.nz);
    if (weno) k_recon_x<true><<<grid, 32 * RW, 0, s>>>(d, par.weno_eps, U, su, Wk, sw, K, sk);
    else k_recon_x<false><<<grid, 32 * RW, 0, s>>>(d, par.mp5_alpha, U, su, Wk, sw, K, sk);
  } else if (weno) launch_march<6, true>(dir, d, par, U, su, Wk, sw, K, sk, fz, s);
  else if (seg == 4) launch_march<4, false>(dir, d, par, U, su, Wk, sw, K, sk, fz, s);
  else if (seg == 6) launch_march<6, false>(dir, d, par, U, su, Wk, sw, K, sk, fz, s);
  else if (seg == 12) launch_march<12, false>(dir, d, par, U, su, Wk, sw, K, sk, fz, s);
  else launch_march<8, false>(dir, d, par, U, su, Wk, sw, K, sk, fz, s);
  return cudaGetLastError();
}

}  // namespace mhd
