// AMR transfer operators on a patch pair: prolongation with the fifth-order Lagrange formula of PAPER.md
// Eq. (80) l.612-620 (1-D operator applied along x, y, z: reading R38), copy restriction (l.626), and the dense-output interpolators
// of Eqs. (56)-(59) l.412-434 used by the Berger-Oliger-without-order-reduction sub-cycling (l.644-649).
//
// Refinement ratio 2, vertex-centred grids: fine interior index a sits at coarse position origin + a/2; even a coincides with a coarse
// point, odd a is a midpoint. All three kernels are streaming passes bound by HBM / L1.
//   k_prolong   a thread owns one coarse x position c and produces the fine pair (2c, 2c+1): the six coarse values c-2..c+3 it loads
//               give both the copy and the Eq. (80) midpoint, so a warp has no parity divergence along x and its loads are
//               coalesced; the y and z parities are uniform per CTA (blockIdx.y/z = fine j, k). Coarse rows are re-read through L1.
//   k_restrict  a thread per coarse target point, stride-2 reads of the fine patch.
//   k_dense     Uout = [U0 +] sum_j c_j K_j on the interior (c_j = dt b_j(theta), or dt^(1-m) d^m b_j / dtheta^m for Eq. 57).
#include "mhd_internal.cuh"

namespace mhd {

namespace {

__device__ __forceinline__ int half_floor(int a) { return a >> 1; }   // arithmetic shift: floor for either sign

struct AxisW { int n, off0; };   // 1 weight at offset 0 (coincident) or 6 weights at offsets -2..3 (Eq. 80)

__device__ __forceinline__ double w80(int m) {   // (3, -25, 150, 150, -25, 3) / 256
  return m == 0 || m == 5 ? 3.0 / 256.0 : (m == 1 || m == 4 ? -25.0 / 256.0 : 150.0 / 256.0);
}

struct ProlongArgs {
  Dims dc, df;
  int origin[3], lo[3], hi[3];
  int c_lo;          // first coarse x position (relative index: fine a = 2 c, 2 c + 1) covered by the box
  int nfields;
};

__global__ void __launch_bounds__(128) k_prolong(const __grid_constant__ ProlongArgs A, const double* __restrict__ Uc, size_t sc,
                                                 double* __restrict__ Uf, size_t sf) {
  const int c = A.c_lo + blockIdx.x * blockDim.x + threadIdx.x;         // coarse position relative to origin (fine a = 2c, 2c+1)
  const int J = A.lo[1] + blockIdx.y, K = A.lo[2] + blockIdx.z;         // fine array indices
  const int Ie = 2 * c + A.df.ng, Io = Ie + 1;                          // fine array x indices of the pair
  const bool we = Ie >= A.lo[0] && Ie < A.hi[0], wo = Io >= A.lo[0] && Io < A.hi[0];
  if (!we && !wo) return;
  const int aj = J - A.df.ng, ak = K - A.df.ng;
  const int cy = A.origin[1] + half_floor(aj) + A.dc.ng, cz = A.origin[2] + half_floor(ak) + A.dc.ng, cx = A.origin[0] + c + A.dc.ng;
  const bool oy = aj & 1, oz = ak & 1;
  const int ny = oy ? 6 : 1, nz = oz ? 6 : 1;
  const size_t pf = (size_t)K * A.df.sz + (size_t)J * A.df.sy;
  for (int f = 0; f < A.nfields; ++f) {
    const double* u = Uc + (size_t)f * sc;
    double se = 0.0, so = 0.0;
    for (int n = 0; n < nz; ++n) {
      const double wz = oz ? w80(n) : 1.0;
      const int z = cz + (oz ? n - 2 : 0);
      double ye = 0.0, yo = 0.0;
      for (int m = 0; m < ny; ++m) {
        const double wy = oy ? w80(m) : 1.0;
        const double* r = u + (size_t)z * A.dc.sz + (size_t)(cy + (oy ? m - 2 : 0)) * A.dc.sy + cx;
        const double u0 = __ldg(r), u1 = __ldg(r + 1);
        ye = fma(wy, u0, ye);
        if (wo) {
          const double um1 = __ldg(r - 1), up2 = __ldg(r + 2), um2 = __ldg(r - 2), up3 = __ldg(r + 3);
          yo = fma(wy, (150.0 * (u0 + u1) - 25.0 * (um1 + up2) + 3.0 * (um2 + up3)) * (1.0 / 256.0), yo);
        }
      }
      se = fma(wz, ye, se);
      so = fma(wz, yo, so);
    }
    double* o = Uf + (size_t)f * sf + pf;
    if (we) o[Ie] = se;
    if (wo) o[Io] = so;
  }
}

struct RestrictArgs { Dims dc, df; int origin[3]; int nfields; };

__global__ void __launch_bounds__(128) k_restrict(const __grid_constant__ RestrictArgs A, const double* __restrict__ Uf, size_t sf,
                                                  double* __restrict__ Uc, size_t sc) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;   // coarse offsets: fine interior (2i, 2j, 2k)
  if (2 * i >= A.df.nx) return;
  const size_t pf = (size_t)(2 * k + A.df.ng) * A.df.sz + (size_t)(2 * j + A.df.ng) * A.df.sy + (2 * i + A.df.ng);
  const size_t pc = (size_t)(A.origin[2] + k + A.dc.ng) * A.dc.sz + (size_t)(A.origin[1] + j + A.dc.ng) * A.dc.sy + (A.origin[0] + i + A.dc.ng);
  for (int f = 0; f < A.nfields; ++f) Uc[(size_t)f * sc + pc] = __ldg(Uf + (size_t)f * sf + pf);
}

struct DenseArgs { const double* K[4]; size_t sk[4]; double c[4]; int nk, with_u0; };

__global__ void __launch_bounds__(128) k_dense(Dims d, int nfields, double* __restrict__ Uout, size_t so, const double* __restrict__ U0, size_t s0,
                                               const __grid_constant__ DenseArgs a) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.nx) return;
  const size_t p = (size_t)(blockIdx.z + d.ng) * d.sz + (size_t)(blockIdx.y + d.ng) * d.sy + (i + d.ng);
  for (int f = 0; f < nfields; ++f) {
    double acc = 0.0;
    for (int m = 0; m < a.nk; ++m) acc = fma(a.c[m], __ldg(a.K[m] + (size_t)f * a.sk[m] + p), acc);
    Uout[(size_t)f * so + p] = a.with_u0 ? __ldg(U0 + (size_t)f * s0 + p) + acc : acc;
  }
}


// ---------------------------------------------------------------------------------------------------------------
// Prolongation of large boxes as three separable passes through shared memory (default when the box is at least a tile in every
// direction): a CTA owns a block of 32 x 8 x 8 fine points whose first point has EVEN fine interior indices, loads the 21 x 9 x 9 coarse
// points under it (block / 2 + the 5 stencil points of Eq. 80) once, and applies the 1-D operator along x (-> 32 x 9 x 9), y (-> 32 x 8 x 9)
// and z (-> 32 x 8 x 8). A fine point then costs ~3.4 one-dimensional evaluations from shared memory instead of up to 6^3 coarse loads.
// ---------------------------------------------------------------------------------------------------------------
constexpr int PFX = 32, PFY = 8, PFZ = 8, PCX = PFX / 2 + 5, PCY = PFY / 2 + 5, PCZ = PFZ / 2 + 5;   // coarse tile 21 x 9 x 9

__device__ __forceinline__ double eq80(const double* u, int s) {          // u points at U_i; midpoint between U_i and U_{i+1}
  return (150.0 * (u[0] + u[s]) - 25.0 * (u[-s] + u[2 * s]) + 3.0 * (u[-2 * s] + u[3 * s])) * (1.0 / 256.0);
}

__global__ void __launch_bounds__(256) k_prolong_tiled(const __grid_constant__ ProlongArgs A, const double* __restrict__ Uc, size_t sc,
                                                       double* __restrict__ Uf, size_t sf, int a0x, int a0y, int a0z) {
  __shared__ double CY[PCZ * PFY * PFX];           // coarse tile (index ((z * PCY) + y) * PCX + x, x = coarse offset + 2), then, once the x pass has consumed it, the result of the y pass
  __shared__ double X[PCZ * PCY * PFX];            // after the x pass
  static_assert(PCZ * PFY * PFX >= PCZ * PCY * PCX, "the y-pass buffer doubles as the coarse tile");
  double* C = CY; double* Y = CY;
  const int tid = threadIdx.x;
  // fine interior indices of the block's first point (even) and the coarse array indices under it
  const int ax = a0x + blockIdx.x * PFX, ay = a0y + blockIdx.y * PFY, az = a0z + blockIdx.z * PFZ;
  const int cx = A.origin[0] + (ax >> 1) + A.dc.ng, cy = A.origin[1] + (ay >> 1) + A.dc.ng, cz = A.origin[2] + (az >> 1) + A.dc.ng;
  for (int f = 0; f < A.nfields; ++f) {
    const double* u = Uc + (size_t)f * sc;
    __syncthreads();                                // the previous field's passes are done with the buffers
    for (int e = tid; e < PCZ * PCY * PCX; e += 256) {
      const int x = e % PCX, y = (e / PCX) % PCY, z = e / (PCX * PCY);
      // clamped: points of a ragged block that fall outside the coarse array feed only fine points outside the box
      const int gx = min(max(cx + x - 2, 0), A.dc.mx - 1), gy = min(max(cy + y - 2, 0), A.dc.my - 1), gz = min(max(cz + z - 2, 0), A.dc.mz - 1);
      C[e] = __ldg(u + (size_t)gz * A.dc.sz + (size_t)gy * A.dc.sy + gx);
    }
    __syncthreads();
    for (int e = tid; e < PCZ * PCY * PFX; e += 256) {             // x pass: fine x index i, even -> copy, odd -> Eq. (80)
      const int i = e % PFX, r = e / PFX;
      const double* c = C + r * PCX + (i >> 1) + 2;
      X[e] = (i & 1) ? eq80(c, 1) : c[0];
    }
    __syncthreads();
    for (int e = tid; e < PCZ * PFY * PFX; e += 256) {             // y pass
      const int i = e % PFX, j = (e / PFX) % PFY, z = e / (PFX * PFY);
      const double* c = X + (z * PCY + (j >> 1) + 2) * PFX + i;
      Y[e] = (j & 1) ? eq80(c, PFX) : c[0];
    }
    __syncthreads();
    double* o = Uf + (size_t)f * sf;
    for (int e = tid; e < PFZ * PFY * PFX; e += 256) {             // z pass and store (x fastest: coalesced)
      const int i = e % PFX, j = (e / PFX) % PFY, k = e / (PFX * PFY);
      const int I = ax + i + A.df.ng, J = ay + j + A.df.ng, K = az + k + A.df.ng;      // fine array indices
      if (I < A.lo[0] || I >= A.hi[0] || J < A.lo[1] || J >= A.hi[1] || K < A.lo[2] || K >= A.hi[2]) continue;
      const double* c = Y + (((k >> 1) + 2) * PFY + j) * PFX + i;
      o[(size_t)K * A.df.sz + (size_t)J * A.df.sy + I] = (k & 1) ? eq80(c, PFY * PFX) : c[0];
    }
  }
}

}  // namespace

cudaError_t launch_prolong(const Dims& dc, const double* Uc, size_t sc, const Dims& df, double* Uf, size_t sf, int nfields,
                           const int origin[3], const int lo[3], const int hi[3], cudaStream_t s) {
  ProlongArgs A;
  A.dc = dc; A.df = df; A.nfields = nfields;
  for (int a = 0; a < 3; ++a) { A.origin[a] = origin[a]; A.lo[a] = lo[a]; A.hi[a] = hi[a]; }
  if (hi[0] <= lo[0] || hi[1] <= lo[1] || hi[2] <= lo[2]) return cudaSuccess;
  auto hf = [](int a) { return a >= 0 ? a / 2 : -((-a + 1) / 2); };
  if (hi[0] - lo[0] >= PFX && hi[1] - lo[1] >= PFY && hi[2] - lo[2] >= PFZ) {
    // blocks anchored at even fine interior indices at or below the box's first point
    const int a0x = 2 * hf(lo[0] - df.ng), a0y = 2 * hf(lo[1] - df.ng), a0z = 2 * hf(lo[2] - df.ng);
    dim3 grid((hi[0] - df.ng - a0x + PFX - 1) / PFX, (hi[1] - df.ng - a0y + PFY - 1) / PFY, (hi[2] - df.ng - a0z + PFZ - 1) / PFZ);
    k_prolong_tiled<<<grid, 256, 0, s>>>(A, Uc, sc, Uf, sf, a0x, a0y, a0z);
    return cudaGetLastError();
  }
  A.c_lo = hf(lo[0] - df.ng);
  const int c_hi = hf(hi[0] - 1 - df.ng);
  dim3 grid((c_hi - A.c_lo + 1 + 127) / 128, hi[1] - lo[1], hi[2] - lo[2]);
  k_prolong<<<grid, 128, 0, s>>>(A, Uc, sc, Uf, sf);
  return cudaGetLastError();
}

cudaError_t launch_restrict(const Dims& df, const double* Uf, size_t sf, const Dims& dc, double* Uc, size_t sc, int nfields, const int origin[3], cudaStream_t s) {
  RestrictArgs A;
  A.dc = dc; A.df = df; A.nfields = nfields;
  for (int a = 0; a < 3; ++a) A.origin[a] = origin[a];
  const int cx = (df.nx + 1) / 2, cy = (df.ny + 1) / 2, cz = (df.nz + 1) / 2;
  dim3 grid((cx + 127) / 128, cy, cz);
  k_restrict<<<grid, 128, 0, s>>>(A, Uf, sf, Uc, sc);
  return cudaGetLastError();
}

cudaError_t launch_dense(const Dims& d, int nfields, double* Uout, size_t so, const double* U0, size_t s0, int nk, const double* const* K,
                         const size_t* sk, const double* c, int with_u0, cudaStream_t s) {
  DenseArgs a;
  a.nk = nk; a.with_u0 = with_u0;
  for (int m = 0; m < 4; ++m) { a.K[m] = m < nk ? K[m] : nullptr; a.sk[m] = m < nk ? sk[m] : 0; a.c[m] = m < nk ? c[m] : 0.0; }
  dim3 grid((d.nx + 127) / 128, d.ny, d.nz);
  k_dense<<<grid, 128, 0, s>>>(d, nfields, Uout, so, U0, s0, a);
  return cudaGetLastError();
}

}  // namespace mhd
