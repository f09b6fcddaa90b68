// a3-a5 (+ a4, a8): CCZ4 + gauge right-hand side, Eqs. (13)-(26) l.141-202, with the 4th-order centred
// differences of Eqs. (60)-(62), the one-sided advective stencils (l.454-456), Kreiss-Oliger dissipation (l.460),
// the matter projections tau, S_i, S_ij (l.188-192, l.260) and — because they need the very same derivatives of
// alpha, beta^i, gamma~_ij, chi — the geometric and divergence-cleaning SOURCES of the GRMHD system (right-hand
// sides of Eq. 32, l.256). Output: K_f for the 22 spacetime fields, and the source part of the 10 fluid fields
// (the flux kernels of flux.cu subtract the flux divergence afterwards).
//
// Two kernels:
//   k_ccz4_algebra  everything that needs the radius-2 centred derivatives (Eqs. 60-62). A CTA owns a 16 x TY x TZ tile, one
//                   point per thread (default 16x4x2 = 128 threads, two CTAs per SM: the derivative phase of one CTA, bound by
//                   shared-memory loads, overlaps the pointwise algebra of the other, bound by the FP64 pipe). The 16 fields
//                   that are differentiated are staged one at a time through a 3-deep shared-memory ring of 22 x (TY+4) x (TZ+4)
//                   tiles (tile + halo) filled by the copy engine (TMA), so every stencil operand is an LDS with a compile-time
//                   offset and the copy of field f+2 overlaps the arithmetic on field f. Phase 1 turns each tile into
//                   derivatives, folds second derivatives, d Gamma^, d K^, d Theta into register accumulators at once
//                   (gamma~^mn d_m d_n gamma~_ab, gamma~^jk d_j d_k beta^c, d_j d_k beta^k, ...) and parks the 33 first
//                   derivatives the algebra needs more than once (NSCR) per point in a per-thread shared-memory scratch column;
//                   phase 2 is the pointwise algebra of Eqs. (13)-(26) and the sources of Eq. (32) reading that scratch.
//   k_adv_ko        beta^k d_k u with the one-sided stencils plus the KO term, radius 3, 1-D along each axis, added to
//                   K for the 22 spacetime fields (and KO alone for the matter fields when sigma_ko_matter != 0).
//                   A thread marches AZ = 4 zones along z with a register window; x / y neighbours come from L1.
//
// All stencils are evaluated on differences (note N1 of DESIGN.md): algebraically identical to the printed
// coefficients, exact zeros in flat space, no cancellation noise.
#include <cuda.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include "mhd_internal.cuh"
#include "tma.cuh"

namespace mhd {

namespace {

__device__ __forceinline__ constexpr int sym(int i, int j) { return i <= j ? (i * (5 - i)) / 2 + j : (j * (5 - j)) / 2 + i; }   // (0,0)=0 (0,1)=1 (0,2)=2 (1,1)=3 (1,2)=4 (2,2)=5

// ------------------------------------------------------------------------------------------------ tile geometry
constexpr int TX = 16, RH = 2;                                        // the tile extents TY, TZ are template parameters of the kernel
// x halo of the shared tile: 3 to the left although the stencil radius is 2. A cp.async.bulk.tensor box must start on a 16-byte boundary
// of global memory (measured on sm_100a: an odd x origin of 8-byte elements raises "illegal instruction"); with ng = 3 ghost points and
// TX even the box that starts 3 points left of the tile does, and 22 x 8 bytes is a whole number of 16-byte units.
constexpr int XL = 3;
constexpr int SX = TX + XL + RH + 1;                                  // shared tile: 22 x (TY + 4) x (TZ + 4)
constexpr int NBUF = 3;
constexpr int OX = 1, OY = SX;                                        // shared-memory strides (z: SX * (TY + 4))

// scratch slots (per thread): only what the pointwise algebra needs more than once. Second derivatives, d Gamma^, d K^ and
// d Theta enter the right-hand side linearly and are folded into register accumulators the moment they are computed.
enum {
  S_DG = 0,       // 18: d_c gamma~_ab at S_DG + 6 c + ab
  S_DDAL = 18,    //  6: d_a d_b alpha
  S_DBE = 24,     //  9: d_a beta^c at S_DBE + 3 a + c
  NSCR = 33
};
template <int TY, int TZ> constexpr size_t smem_bytes() { return (size_t)(NBUF * ((SX * (TY + 2 * RH) * (TZ + 2 * RH) + 15) & ~15) + NSCR * TX * TY * TZ) * sizeof(double) + 128; }   // + mbarriers

__device__ __forceinline__ void cp_async8(double* smem, const double* gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// ---- TMA: one cp.async.bulk.tensor per field and tile (a 22 x (TY+4) x (TZ+4) box of the 4-D tensor (x, y, z, field); coordinates past the end of
// the array are zero-filled by the copy engine: those points belong to ragged tiles and are masked), completion on an mbarrier: tma.cuh

// unscaled Eq. (60): 12 h D u
template <int O>
__device__ __forceinline__ double d1u(const double* s) { return 8.0 * (s[O] - s[-O]) - (s[2 * O] - s[-2 * O]); }
// unscaled Eq. (62): 12 h^2 D^2 u, on differences from the centre
template <int O>
__device__ __forceinline__ double d2u(const double* s, double u0) {
  return 16.0 * ((s[O] - u0) + (s[-O] - u0)) - ((s[2 * O] - u0) + (s[-2 * O] - u0));
}
// unscaled Eq. (61): 144 h_a h_b D_b (D_a u)
template <int OA, int OB>
__device__ __forceinline__ double d11u(const double* s) {
  return 8.0 * (d1u<OA>(s + OB) - d1u<OA>(s - OB)) - (d1u<OA>(s + 2 * OB) - d1u<OA>(s - 2 * OB));
}

struct Scale { double i12h[3], i12h2[3], i144[3]; };   // i144: xy, xz, yz

template <int OZ>
__device__ __forceinline__ void first(const double* s, const Scale& sc, double o[3]) {
  o[0] = d1u<OX>(s) * sc.i12h[0]; o[1] = d1u<OY>(s) * sc.i12h[1]; o[2] = d1u<OZ>(s) * sc.i12h[2];
}
// second derivatives in sym order xx, xy, xz, yy, yz, zz
template <int OZ>
__device__ __forceinline__ void second(const double* s, const Scale& sc, double o[6]) {
  const double u0 = s[0];
  o[0] = d2u<OX>(s, u0) * sc.i12h2[0]; o[3] = d2u<OY>(s, u0) * sc.i12h2[1]; o[5] = d2u<OZ>(s, u0) * sc.i12h2[2];
  o[1] = d11u<OX, OY>(s) * sc.i144[0]; o[2] = d11u<OX, OZ>(s) * sc.i144[1]; o[4] = d11u<OY, OZ>(s) * sc.i144[2];
}

}  // namespace

// order in which the differentiated fields pass through the ring
__device__ constexpr int FORDER[16] = {GXX, GXY, GXZ, GYY, GYZ, GZZ, GAMX, GAMY, GAMZ, CHI, ALPHA, BETAX, BETAY, BETAZ, KHAT, THETA};

template <int TY, int TZ, bool TMA>
__global__ void __launch_bounds__(TX * TY * TZ, (TX * TY * TZ <= 64 ? 4 : TX * TY * TZ <= 128 ? 2 : 1))
k_ccz4_algebra(const __grid_constant__ Dims d, const __grid_constant__ Par par, const double* __restrict__ U, size_t su,
               const double* __restrict__ P, size_t sp, double* __restrict__ K, size_t sk, const __grid_constant__ CUtensorMap tmap) {
  constexpr int SY = TY + 2 * RH, OZ = SX * SY;
  constexpr int SZ = TZ + 2 * RH, TILE = SX * SY * SZ, NT = TX * TY * TZ, NLD = TMA ? 1 : (TILE + NT - 1) / NT;
  constexpr int TILEP = (TILE + 15) & ~15;             // buffer stride: TMA destination tiles must stay 128-byte aligned
  extern __shared__ __align__(128) double smem[];
  double* ring = smem;
  const int tid = threadIdx.x;
  double* scr = smem + NBUF * TILEP + tid;
  uint64_t* full = (uint64_t*)(smem + NBUF * TILEP + NSCR * NT);   // NBUF mbarriers (TMA path)
#define SCR(slot) scr[(slot) * NT]
  const int tx = tid % TX, ty = (tid / TX) % TY, tz = tid / (TX * TY);
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY, k0 = blockIdx.z * TZ;
  const int i = i0 + tx, j = j0 + ty, k = k0 + tz;
  const bool inside = i < d.nx && j < d.ny && k < d.nz;
  // centre point (clamped for the threads of a ragged tile: they take part in the copies and barriers only)
  const size_t pt = (size_t)(min(k, d.nz - 1) + d.ng) * d.sz + (size_t)(min(j, d.ny - 1) + d.ng) * d.sy + (min(i, d.nx - 1) + d.ng);

  // cp.async path: global offsets of the NLD tile elements this thread copies (clamped into the ghosted array)
  int goff[NLD];
  if (!TMA) {
#pragma unroll
    for (int m = 0; m < NLD; ++m) {
      const int e = min(tid + m * NT, TILE - 1);
      const int x = e % SX, y = (e / SX) % SY, z = e / (SX * SY);
      const int gx = min(i0 + x - XL + d.ng, d.mx - 1), gy = min(j0 + y - RH + d.ng, d.my - 1), gz = min(k0 + z - RH + d.ng, d.mz - 1);
      goff[m] = (int)(gz * d.sz + gy * d.sy + gx);
    }
  } else {
    if (tid == 0) {
#pragma unroll
      for (int b = 0; b < NBUF; ++b) mbar_init(full + b, 1);
      mbar_fence_init();
    }
    __syncthreads();
  }
  auto issue = [&](int f, int buf) {
    if (TMA) {                                           // one thread arms the barrier and hands the box to the copy engine
      if (tid == 0) {
        mbar_expect_tx(full + buf, TILE * (unsigned)sizeof(double));
        tma_load_4d(ring + buf * TILEP, &tmap, full + buf, i0 - XL + d.ng, j0 - RH + d.ng, k0 - RH + d.ng, f);
      }
    } else {
      const double* src = U + (size_t)f * su;
      double* dst = ring + buf * TILEP + tid;
#pragma unroll
      for (int m = 0; m < NLD; ++m) if (TILE % NT == 0 || tid + m * NT < TILE) cp_async8(dst + m * NT, src + goff[m]);
      cp_commit();
    }
  };
  issue(FORDER[0], 0);
  issue(FORDER[1], 1);

  Scale sc;
  {
    const double h[3] = {d.dx, d.dy, d.dz};
#pragma unroll
    for (int a = 0; a < 3; ++a) { sc.i12h[a] = 1.0 / (12.0 * h[a]); sc.i12h2[a] = 1.0 / (12.0 * h[a] * h[a]); }
    sc.i144[0] = sc.i12h[0] * sc.i12h[1]; sc.i144[1] = sc.i12h[0] * sc.i12h[2]; sc.i144[2] = sc.i12h[1] * sc.i12h[2];
  }
  auto F = [&](int f) { return __ldg(U + (size_t)f * su + pt); };

  // ---- point values of the conformal metric and its inverse (needed to contract second derivatives in phase 1)
  double g[6], gi[6];
#pragma unroll
  for (int a = 0; a < 6; ++a) g[a] = F(GXX + a);
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
#define G_(i, j) g[sym(i, j)]
#define GI(i, j) gi[sym(i, j)]

  // The pointwise phase reads 21 point values that are not in the ring (A~_ij, the 10 conserved fluid fields, W, p, v^i). There are no registers to
  // hold them through phase 1 and only two warps per scheduler to cover an HBM latency each, so the lines are pulled into L1 now
  // and the loads of phase 2 find them there.
  {
    auto pf = [](const double* a) { asm volatile("prefetch.global.L1 [%0];" ::"l"(a)); };
#pragma unroll
    for (int a = 0; a < 6; ++a) pf(U + (size_t)(AXX + a) * su + pt);
#pragma unroll
    for (int a = 0; a < 10; ++a) pf(U + (size_t)(DBAR + a) * su + pt);
    pf(P + (size_t)WLOR * sp + pt); pf(P + (size_t)PRESS * sp + pt);
#pragma unroll
    for (int a = 0; a < 3; ++a) pf(P + (size_t)(VX + a) * sp + pt);
  }

  // ================================================================= phase 1: derivatives, field by field
  const int ctr = ((tz + RH) * SY + (ty + RH)) * SX + (tx + XL);
  const double chi = F(CHI), al = F(ALPHA);
  double be[3] = {0, 0, 0}, Gh[3] = {0, 0, 0}, Kh = 0.0, Th = 0.0;
  double Racc[6] = {0, 0, 0, 0, 0, 0};   // part of chi (R^_ab + R^chi_ab) that is linear in second derivatives and in d Gamma^
  double GamAcc[3] = {0, 0, 0};          // gamma~^jk d_j d_k beta^a + 1/3 gamma~^ab d_b d_k beta^k - 2 alpha gamma~^ab (2/3 d_b K^ + 1/3 d_b Theta)
  double dchi[3] = {0, 0, 0}, dal[3] = {0, 0, 0};
#pragma unroll
  for (int n = 0; n < 16; ++n) {
    if (TMA) {
      __syncthreads();                                   // everybody is done reading the buffer the next copy overwrites
      if (n + 2 < 16) issue(FORDER[n + 2], (n + 2) % NBUF);
      mbar_wait(full + n % NBUF, (n / NBUF) & 1);        // field n has landed (the barrier of a buffer completes once per use)
    } else {
      if (n + 1 < 16) cp_wait<1>(); else cp_wait<0>();
      __syncthreads();
      if (n + 2 < 16) issue(FORDER[n + 2], (n + 2) % NBUF);
    }
    const double* s = ring + (n % NBUF) * TILEP + ctr;
    double d1[3];
    first<OZ>(s, sc, d1);
    if (n < 6) {                       // gamma~_ab, ab = n: -1/2 gamma~^mn d_m d_n gamma~_ab of Eq. (23)
      double dd[6];
      second<OZ>(s, sc, dd);
#pragma unroll
      for (int c = 0; c < 3; ++c) SCR(S_DG + 6 * c + n) = d1[c];
      Racc[n] -= chi * (0.5 * (gi[0] * dd[0] + gi[3] * dd[3] + gi[5] * dd[5]) + (gi[1] * dd[1] + gi[2] * dd[2] + gi[4] * dd[4]));
    } else if (n < 9) {                // Gamma^^c, c = n - 6: gamma~_k(i d_j) Gamma^^k
      const int c = n - 6;
      Gh[c] = s[0];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) Racc[sym(a, b)] += 0.5 * chi * (G_(c, a) * d1[b] + G_(c, b) * d1[a]);
    } else if (n == 9) {               // chi: 1/2 d_i d_j chi + 1/2 gamma~_ij gamma~^mn d_m d_n chi of Eq. (22)
      double dd[6];
      second<OZ>(s, sc, dd);
      const double lap = gi[0] * dd[0] + gi[3] * dd[3] + gi[5] * dd[5] + 2.0 * (gi[1] * dd[1] + gi[2] * dd[2] + gi[4] * dd[4]);
#pragma unroll
      for (int a = 0; a < 3; ++a) dchi[a] = d1[a];
#pragma unroll
      for (int a = 0; a < 6; ++a) Racc[a] += 0.5 * dd[a] + 0.5 * g[a] * lap;
    } else if (n == 10) {              // alpha
      double dd[6];
      second<OZ>(s, sc, dd);
#pragma unroll
      for (int a = 0; a < 3; ++a) dal[a] = d1[a];
#pragma unroll
      for (int a = 0; a < 6; ++a) SCR(S_DDAL + a) = dd[a];
    } else if (n < 14) {               // beta^c, c = n - 11
      const int c = n - 11;
      double dd[6];
      second<OZ>(s, sc, dd);
      be[c] = s[0];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        SCR(S_DBE + 3 * a + c) = d1[a];
        GamAcc[a] += (1.0 / 3.0) * (GI(a, 0) * dd[sym(0, c)] + GI(a, 1) * dd[sym(1, c)] + GI(a, 2) * dd[sym(2, c)]);
      }
      GamAcc[c] += gi[0] * dd[0] + gi[3] * dd[3] + gi[5] * dd[5] + 2.0 * (gi[1] * dd[1] + gi[2] * dd[2] + gi[4] * dd[4]);
    } else {                           // K^ (weight 2/3), Theta (weight 1/3): -2 alpha gamma~^ab w d_b
      if (n == 14) Kh = s[0]; else Th = s[0];
      const double w = -2.0 * al * (n == 14 ? 2.0 / 3.0 : 1.0 / 3.0);
#pragma unroll
      for (int a = 0; a < 3; ++a) GamAcc[a] += w * (GI(a, 0) * d1[0] + GI(a, 1) * d1[1] + GI(a, 2) * d1[2]);
    }
  }
  if (!inside) return;
  (void)be;

  // ================================================================= phase 2: pointwise algebra
  auto OUT = [&](int f) -> double& { return K[(size_t)f * sk + pt]; };
  const double ichi = 1.0 / chi;

  // ---- Christoffels of the conformal metric: Gl[k][ij] = Gamma~_kij, Gu[k][ij] = Gamma~^k_ij
  double Gl[3][6], Gu[3][6], Gt[3];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b)
        Gl[c][sym(a, b)] = 0.5 * (SCR(S_DG + 6 * a + sym(c, b)) + SCR(S_DG + 6 * b + sym(c, a)) - SCR(S_DG + 6 * c + sym(a, b)));
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int a = 0; a < 6; ++a) Gu[c][a] = GI(c, 0) * Gl[0][a] + GI(c, 1) * Gl[1][a] + GI(c, 2) * Gl[2][a];
#pragma unroll
  for (int c = 0; c < 3; ++c)
    Gt[c] = gi[0] * Gu[c][0] + gi[3] * Gu[c][3] + gi[5] * Gu[c][5] + 2.0 * (gi[1] * Gu[c][1] + gi[2] * Gu[c][2] + gi[4] * Gu[c][4]);
  double Z[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) Z[c] = 0.5 * chi * (Gh[c] - Gt[c]);          // l.132

  // ---- chi R^_ij  (Eq. 23 times chi), accumulated component by component
  double X[6];   // becomes alpha (chi R^_ij + chi R^chi_ij - 8 pi G chi S_ij) - chi D_i D_j alpha
  // gamma~^mn (2 Gamma~^c_m(a Gamma~_b)cn + Gamma~^c_am Gamma~_cnb) with the contraction over m done once: H[c][n][a] = gamma~^mn Gamma~^c_ma
  // (81 + 162 multiply-adds instead of 540)
  double H[3][3][3];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int n = 0; n < 3; ++n)
#pragma unroll
      for (int a = 0; a < 3; ++a) H[c][n][a] = GI(0, n) * Gu[c][sym(0, a)] + GI(1, n) * Gu[c][sym(1, a)] + GI(2, n) * Gu[c][sym(2, a)];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = a; b < 3; ++b) {
      const int ab = sym(a, b);
      double r = 0.0;
#pragma unroll
      for (int c = 0; c < 3; ++c) r += 0.5 * Gh[c] * (Gl[a][sym(b, c)] + Gl[b][sym(a, c)]);        // Gamma^^k Gamma~_(ij)k
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int n = 0; n < 3; ++n)
          r += H[c][n][a] * (Gl[b][sym(c, n)] + Gl[c][sym(n, b)]) + H[c][n][b] * Gl[a][sym(c, n)];
      X[ab] = Racc[ab] + chi * r;
    }
  double Rtr = 0.0;   // gamma^ij (R_ij + 2 D_(i Z_j)) = gamma~^ij (chi R^_ij + chi R^chi_ij)

  // ---- chi R^chi_ij (Eq. 22), physical Hessian of the lapse (R25)
  double gdchi[3];   // gamma~^kl d_l chi
#pragma unroll
  for (int c = 0; c < 3; ++c) gdchi[c] = GI(c, 0) * dchi[0] + GI(c, 1) * dchi[1] + GI(c, 2) * dchi[2];
  double lapal;      // D_i D^i alpha, Eq. (24)
  {
    double ddal[6];
#pragma unroll
    for (int a = 0; a < 6; ++a) ddal[a] = SCR(S_DDAL + a);
    double lapchi = 0.0, Ghdchi = 0.0, Zl[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      Ghdchi += Gh[a] * dchi[a];
      Zl[a] = G_(a, 0) * Z[0] + G_(a, 1) * Z[1] + G_(a, 2) * Z[2];        // Z^k gamma~_ka
#pragma unroll
      for (int b = 0; b < 3; ++b) lapchi -= GI(a, b) * 1.5 * ichi * dchi[a] * dchi[b];   // its second-derivative part is in Racc
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
        double c_ = -0.25 * ichi * dchi[a] * dchi[b];
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
  // ---- matter (l.188-192, l.260)
  const double G8 = 8.0 * 3.14159265358979323846 * par.grav_G;
  const double isg = chi * sqrt(chi);   // 1/sqrt(gamma)
  double uc[10];
#pragma unroll
  for (int a = 0; a < 10; ++a) uc[a] = F(DBAR + a);
  double Sij[6];   // undensitised S_ij, l.260
  double E, Sl[3];
  {
    const double W = __ldg(P + (size_t)WLOR * sp + pt), pr = __ldg(P + (size_t)PRESS * sp + pt);
    double vu[3], vl[3], Bu[3], Bl[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) { vu[a] = __ldg(P + (size_t)(VX + a) * sp + pt); Bu[a] = uc[6 + a] * isg; Sl[a] = uc[3 + a] * isg; }
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
    for (int c = 0; c < 3; ++c) dbe[a][c] = SCR(S_DBE + 3 * a + c);
  const double divb = dbe[0][0] + dbe[1][1] + dbe[2][2];

  // ---- curvature fields
  double A[6];
#pragma unroll
  for (int a = 0; a < 6; ++a) A[a] = F(AXX + a);
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

  const double logdet = log(detg);
  // ---- Eq. (13) without the advective / KO part (k_adv_ko adds it)
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = a; b < 3; ++b) {
      const int ab = sym(a, b);
      double s = 0.0;
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
      double s = 0.0, AAab = 0.0;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        s += A[sym(a, c)] * dbe[b][c] + A[sym(c, b)] * dbe[a][c];
        AAab += A[sym(a, c)] * Aud[c][b];
      }
      s += -(2.0 / 3.0) * A[ab] * divb - al * (1.0 / 3.0) * par.kappa_c * g[ab] * trA + X[ab] + al * (Kh * A[ab] - 2.0 * AAab);
      OUT(AXX + ab) = s;
    }
  // ---- Eq. (15)
  OUT(CHI) = (2.0 / 3.0) * chi * (al * Ktot - divb);
  // ---- Eqs. (16), (17)
  const double Zdal = Z[0] * dal[0] + Z[1] * dal[1] + Z[2] * dal[2];
  OUT(KHAT) = -lapal + al * (Ktot * Ktot * (1.0 / 3.0) + AA + 0.5 * G8 * (E + Str) + par.kappa_z * (1.0 - par.kappa_2) * Th) + 2.0 * Zdal;
  OUT(THETA) = 0.5 * al * (Rtr + (2.0 / 3.0) * Kh * Kh + (2.0 / 3.0) * Th * (Kh - 2.0 * Th) - AA) - Zdal
               - al * (G8 * E + par.kappa_z * (2.0 + par.kappa_2) * Th);
  // ---- Eqs. (18)-(20)
  {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      double s = (2.0 / 3.0) * Gh[a] * divb + GamAcc[a];
      double b1 = 0.0, b2 = 0.0;
#pragma unroll
      for (int b = 0; b < 3; ++b) {
        s += -Gh[b] * dbe[b][a] - 2.0 * Auu[sym(a, b)] * dal[b];
#pragma unroll
        for (int c = 0; c < 3; ++c) b1 += Gu[a][sym(b, c)] * Auu[sym(b, c)];
        b1 += -1.5 * ichi * Auu[sym(a, b)] * dchi[b] - G8 * GI(a, b) * Sl[b];
        b2 -= GI(a, b) * (Th / al * dal[b]);
      }
      b2 -= Z[a] * ichi * (par.kappa_z + (2.0 / 3.0) * Ktot);
      OUT(GAMX + a) = s + 2.0 * al * (b1 + b2);
    }
  }
  // ---- gauge, Eqs. (25)-(26)
  OUT(ALPHA) = -2.0 * al * par.f_alpha * Kh;
#pragma unroll
  for (int a = 0; a < 3; ++a) OUT(BETAX + a) = 0.75 * par.f_beta * Gh[a] - par.eta_shift * (be[a] - par.beta0[a]);

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
  }
#undef G_
#undef GI
#undef SCR
}

// ---------------------------------------------------------------------------------------------------------------
// beta^k D_k u (one-sided 4th-order stencils of l.454-456) + KO (l.460), added to K.
// With p_n = u_{i+n} - u_i, m_n = u_{i-n} - u_i the two one-sided stencils are
//     12 h D^+ u = p3 - 6 p2 + 18 p1 - 3 m1 = (Q + A)/2,      12 h D^- u = -(m3 - 6 m2 + 18 m1 - 3 p1) = (A - Q)/2,
//     Q = (p3 + m3) - 6 (p2 + m2) + 15 (p1 + m1)   (the KO combination itself),   A = (p3 - m3) - 6 (p2 - m2) + 21 (p1 - m1),
// so  beta D^{sign beta} u + sigma Q / (64 h) = beta A / (24 h) + (|beta| / (24 h) + sigma / (64 h)) Q :
// no branch on the sign of beta (R15: the two branches agree at beta = 0), one pass over the six differences.
// ---------------------------------------------------------------------------------------------------------------
namespace {

template <bool ADV>
__device__ __forceinline__ double adv_ko_axis(double um3, double um2, double um1, double u0, double up1, double up2, double up3, double cbh, double cko) {
  const double q = ((up3 - u0) + (um3 - u0)) - 6.0 * ((up2 - u0) + (um2 - u0)) + 15.0 * ((up1 - u0) + (um1 - u0));
  if (!ADV) return cko * q;
  const double a = (up3 - um3) - 6.0 * (up2 - um2) + 21.0 * (up1 - um1);
  return fma(cko + fabs(cbh), q, cbh * a);
}

template <bool ADV, int AZ, int MINB, bool FUSED>
__global__ void __launch_bounds__(256, MINB) k_adv_ko(const __grid_constant__ Dims d, double sigma, int f0, int nf,
                                                      const double* __restrict__ U, size_t su, double* __restrict__ K, size_t sk,
                                                      const __grid_constant__ Fuse fz) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 8 + threadIdx.y, k0 = blockIdx.z * AZ;
  if (i >= d.nx || j >= d.ny) return;
  const int nzl = min(AZ, d.nz - k0);
  const int sy = (int)d.sy, sz = (int)d.sz;        // 32-bit strides: neighbour offsets relative to the thread's point stay far below 2^31 (checked at launch)
  const size_t base = (size_t)(k0 + d.ng) * d.sz + (size_t)(j + d.ng) * d.sy + (i + d.ng);
  const double i24h[3] = {1.0 / (24.0 * d.dx), 1.0 / (24.0 * d.dy), 1.0 / (24.0 * d.dz)};
  const double cko[3] = {sigma / (64.0 * d.dx), sigma / (64.0 * d.dy), sigma / (64.0 * d.dz)};
  double cb[AZ][3];   // beta^a / (24 h_a) on the AZ planes
#pragma unroll
  for (int kk = 0; kk < AZ; ++kk)
#pragma unroll
    for (int a = 0; a < 3; ++a) cb[kk][a] = (ADV && kk < nzl) ? __ldg(U + (size_t)(BETAX + a) * su + base + kk * sz) * i24h[a] : 0.0;
#pragma unroll 1
  for (int f = f0; f < f0 + nf; ++f) {
    const double* u = U + (size_t)f * su + base;
    double* ko = K + (size_t)f * sk + base;
    double w[AZ + 6];   // the z column k0-3 .. k0+AZ+2 (clamped for a ragged last block: those planes are not used)
#pragma unroll
    for (int n = 0; n < AZ + 6; ++n) w[n] = __ldg(u + min(n - 3, nzl + 2) * sz);
    double kold[AZ];    // K is read-modify-write: its loads are issued with the stencil loads, not after the arithmetic
#pragma unroll
    for (int kk = 0; kk < AZ; ++kk) kold[kk] = kk < nzl ? ko[kk * sz] : 0.0;
    double pre[AZ];     // U0 + earlier stages of the fused RK combine, fetched with the rest
#pragma unroll
    for (int kk = 0; kk < AZ; ++kk) pre[kk] = (FUSED && kk < nzl) ? fused_fetch(fz, f, base + kk * sz) : 0.0;
#pragma unroll
    for (int kk = 0; kk < AZ; ++kk) {
      if (kk < nzl) {
        const double* c = u + kk * sz;
        const double u0 = w[kk + 3];
        double acc = adv_ko_axis<ADV>(w[kk], w[kk + 1], w[kk + 2], u0, w[kk + 4], w[kk + 5], w[kk + 6], cb[kk][2], cko[2]);
        acc += adv_ko_axis<ADV>(__ldg(c - 3), __ldg(c - 2), __ldg(c - 1), u0, __ldg(c + 1), __ldg(c + 2), __ldg(c + 3), cb[kk][0], cko[0]);
        acc += adv_ko_axis<ADV>(__ldg(c - 3 * sy), __ldg(c - 2 * sy), __ldg(c - sy), u0, __ldg(c + sy), __ldg(c + 2 * sy), __ldg(c + 3 * sy), cb[kk][1], cko[1]);
        if (FUSED) fused_store(fz, f, base + kk * sz, pre[kk], kold[kk] + acc, ko + kk * sz); else ko[kk * sz] = kold[kk] + acc;
      }
    }
  }
}
}  // namespace

// Tensor map of the state slot with the algebra kernel's box: legal for even MX / stride and an even box origin i0 - XL + ng (ng odd);
// otherwise the cp.async path is used. MHD_CCZ4_TMA=0 forces the cp.async path.
static bool make_tensor_map(const Dims& d, const double* U, size_t su, int ty, int tz, CUtensorMap* out) {
  static int off = -1;
  if (off < 0) { const char* v = getenv("MHD_CCZ4_TMA"); off = v && atoi(v) == 0; }
  if (off || ((d.ng - XL) & 1)) return false;
  return make_tensor_map_4d(d, U, su, MHD_NSTATE, SX, ty + 2 * RH, tz + 2 * RH, out);
}

template <int TY, int TZ>
static cudaError_t launch_algebra_tz(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* K, size_t sk, cudaStream_t s) {
  // the opt-in to > 48 KB of dynamic shared memory is per device and per instantiation
  static int attr_set[64][2] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  CUtensorMap map;
  const bool tma = make_tensor_map(d, U, su, TY, TZ, &map);
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  constexpr int SMEM = (int)smem_bytes<TY, TZ>();
  if (!attr_set[dev][tma]) {
    e = tma ? cudaFuncSetAttribute(k_ccz4_algebra<TY, TZ, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM)
            : cudaFuncSetAttribute(k_ccz4_algebra<TY, TZ, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
    if (e != cudaSuccess) return e;
    attr_set[dev][tma] = 1;                              // only after the attribute call succeeded
  }
  const dim3 grid((d.nx + TX - 1) / TX, (d.ny + TY - 1) / TY, (d.nz + TZ - 1) / TZ);
  if (tma) k_ccz4_algebra<TY, TZ, true><<<grid, TX * TY * TZ, SMEM, s>>>(d, par, U, su, P, sp, K, sk, map);
  else {
    memset(&map, 0, sizeof(map));
    k_ccz4_algebra<TY, TZ, false><<<grid, TX * TY * TZ, SMEM, s>>>(d, par, U, su, P, sp, K, sk, map);
  }
  e = cudaGetLastError();
  if (e != cudaSuccess && getenv("MHD_DEBUG")) fprintf(stderr, "libmhd_b200: k_ccz4_algebra<%d, %d, %d> launch: %s\n", TY, TZ, (int)tma, cudaGetErrorString(e));
  return e;
}

// Tile shapes (x extent 16): MHD_CCZ4_TILE = "TYxTZ". 4x2 = 128 threads, two CTAs per SM (default: the derivative phase of one CTA, bound by
// shared-memory loads, overlaps the pointwise algebra of the other, bound by the FP64 pipe); 4x4 = 256 threads, one CTA per SM (round 1);
// 2x2 and 4x1 = 64 threads, four CTAs per SM.
cudaError_t launch_ccz4_algebra(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* K, size_t sk, cudaStream_t s) {
  static int tile = 0;
  if (tile == 0) { const char* v = getenv("MHD_CCZ4_TILE"); tile = v && strlen(v) == 3 ? (v[0] - '0') * 10 + (v[2] - '0') : 42; }
  if (tile == 44) return launch_algebra_tz<4, 4>(d, par, U, su, P, sp, K, sk, s);
  if (tile == 22) return launch_algebra_tz<2, 2>(d, par, U, su, P, sp, K, sk, s);
  if (tile == 41) return launch_algebra_tz<4, 1>(d, par, U, su, P, sp, K, sk, s);
  if (tile == 24) return launch_algebra_tz<2, 4>(d, par, U, su, P, sp, K, sk, s);
  return launch_algebra_tz<4, 2>(d, par, U, su, P, sp, K, sk, s);
}

cudaError_t launch_adv_ko(const Dims& d, const Par& par, const double* U, size_t su, double* K, size_t sk, const Fuse& fz, cudaStream_t s) {
  constexpr int AZ = 4;
  if (d.sz > (1ll << 26)) return cudaErrorInvalidValue;      // the kernel keeps neighbour offsets (up to AZ + 3 planes) in 32 bits
  dim3 ablock(32, 8), agrid((d.nx + 31) / 32, (d.ny + 7) / 8, (d.nz + AZ - 1) / AZ);
  if (fz.Uout) k_adv_ko<true, AZ, 2, true><<<agrid, ablock, 0, s>>>(d, par.sigma_ko_spacetime, 0, 22, U, su, K, sk, fz);   // last kernel to touch the spacetime K
  else k_adv_ko<true, AZ, 3, false><<<agrid, ablock, 0, s>>>(d, par.sigma_ko_spacetime, 0, 22, U, su, K, sk, fz);
  if (par.sigma_ko_matter != 0.0)                                          // R16: optional KO on the matter fields (the fluid K is finished by flux.cu)
    k_adv_ko<false, AZ, 4, false><<<agrid, ablock, 0, s>>>(d, par.sigma_ko_matter, DBAR, 10, U, su, K, sk, fz);
  return cudaGetLastError();
}

}  // namespace mhd
