// Internal declarations of libmhd_b200 (CUDA, sm_100a). Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>
#include "../../include/mhd.h"

namespace mhd {

// field indices of the state and primitive slots (see include/mhd.h)
enum {
  GXX = 0, GXY, GXZ, GYY, GYZ, GZZ, AXX, AXY, AXZ, AYY, AYZ, AZZ, CHI, KHAT, THETA, GAMX, GAMY, GAMZ,
  ALPHA, BETAX, BETAY, BETAZ, DBAR, DYEBAR, TAUBAR, SXBAR, SYBAR, SZBAR, BXBAR, BYBAR, BZBAR, PHIBAR
};
enum { RHO = 0, YE, EPS, PRESS, VX, VY, VZ, WLOR, TEMP, CS2 };

struct Dims {
  int nx, ny, nz, ng, mx, my, mz;
  long long sy, sz;          // strides of j and k in elements
  long long npts;            // mx*my*mz
  double dx, dy, dz;
};

// device-side parameter block, passed by value as a __grid_constant__ kernel argument
struct Par {
  int eos_kind, n_pieces;
  double eos_gamma, eos_gamma_th;
  double pp_K[MHD_MAX_PIECES], pp_Gamma[MHD_MAX_PIECES], pp_rho[MHD_MAX_PIECES], pp_a[MHD_MAX_PIECES];
  const double *tab_logp, *tab_loge, *tab_cs2;
  int n_rho, n_T, n_ye;
  double lr0, dlr, lT0, dlT, ye0, dye, tab_eps_shift, tab_h0;
  double idlr, idlT, idye, tab_rho_lo, tab_rho_hi;   // derived at create time: reciprocal spacings, density range of the table
  double kappa_z, kappa_c, kappa_2, eta_shift, f_alpha, f_beta, beta0[3], grav_G;
  double sigma_ko_spacetime, sigma_ko_matter;
  double c_b, kappa_b, mp5_alpha;
  double rho_atmo, rho_cut, rho_low, alpha_bh, w_max, rho_max, eps_min, eps_max;
  double ye_min, ye_max, ye_atmo, eps_atmo, T_atmo;
  int c2p_maxit;
  double m1_kappa0, m1_rho0, m1_species_scale[3], m1_efloor, m1_tol, m1_mb;
  int m1_maxit, m1_odd_even;
  double m1_arad, m1_oe_guard;
  int recon_kind;
  double weno_eps, les_C_M, les_C_N, les_C_Y, les_C_T;
};

struct Slot {
  void* ptr = nullptr;
  size_t stride = 0;
  // halo exchange fused with the ghost fill: the same slot of the neighbouring patch in direction (dx+1) + 3 (dy+1) + 9 (dz+1)
  // (device pointers, possibly peer-GPU mappings). They travel with the slot when mhd_advance swaps state buffers: every patch of a
  // decomposition performs the same swaps.
  const double* peer[27] = {};
  size_t peer_stride[27] = {};
};

// Explicit RK combine (Eq. 53) fused into the last kernel that touches a field of K_i (k_adv_ko for the 22 spacetime fields,
// k_recon_march<z> for the 10 fluid fields):  Uout = U0 + sum_m cp[m] Kp[m] + cself K_i,  with cp, cself already multiplied by dt.
// Uout must not be the state the stencils read. K_i itself is written only if write_k (the last stage has no later reader).
struct Fuse {
  double* Uout = nullptr; size_t so = 0;          // nullptr: no fused combine (K_i is written)
  const double* U0 = nullptr; size_t s0 = 0;
  const double* Kp[MHD_MAX_STAGES - 1] = {}; size_t skp[MHD_MAX_STAGES - 1] = {}; double cp[MHD_MAX_STAGES - 1] = {};
  int nk = 0;
  double cself = 0.0;
  int write_k = 1;
};
// Two halves, so that the loads are issued with the stencil loads of the kernel and not after its arithmetic:
// fused_fetch returns U0 + sum_m cp[m] Kp[m] at the point, fused_store adds cself K_i and writes.
__device__ __forceinline__ double fused_fetch(const Fuse& fz, int field, size_t pt) {
  if (!fz.Uout) return 0.0;
  double acc = __ldg(fz.U0 + (size_t)field * fz.s0 + pt);
  for (int m = 0; m < fz.nk; ++m) acc = fma(fz.cp[m], __ldg(fz.Kp[m] + (size_t)field * fz.skp[m] + pt), acc);
  return acc;
}
__device__ __forceinline__ void fused_store(const Fuse& fz, int field, size_t pt, double fetched, double knew, double* kdst) {
  if (fz.Uout) {
    fz.Uout[(size_t)field * fz.so + pt] = fma(fz.cself, knew, fetched);
    if (!fz.write_k) return;
  }
  *kdst = knew;
}

}  // namespace mhd

struct mhd_patch {
  mhd_patch_desc desc;
  mhd::Dims dims;
  mhd::Par par;
  mhd::Slot slot[MHD_NSLOTS];
  unsigned long long* d_counts;   // device scratch: 8 counters for mhd_patch_status, then 8 doubles (EoS part of the atmosphere state),
                                  // then [16..42] the 27 halo epoch words of this patch, [43] the halo time-out flag
  unsigned long long* peer_word[27] = {};   // where to signal the neighbour in direction q (its epoch word for direction 26 - q)
  unsigned long long halo_epoch = 0;
  // optional per-kernel timing (mhd_patch_profile)
  bool profiling = false;
  struct Ev { cudaEvent_t a, b; int cls; };
  std::vector<Ev> events;         // recorded pairs since the last read
  std::vector<Ev> pool;           // recycled events
};

namespace mhd {
// kernel launchers (one per translation unit); all return cudaGetLastError()
cudaError_t launch_fill_ghosts(const Dims& d, double* U, size_t stride, int nfields, const int bc[6], const Slot* peers, cudaStream_t s);
cudaError_t launch_halo_signal(unsigned long long* const* words, int n, unsigned long long epoch, cudaStream_t s);
cudaError_t launch_halo_wait(unsigned long long* const* words, int n, unsigned long long epoch, unsigned long long* timeout_flag, cudaStream_t s);
cudaError_t launch_con2prim(const Dims& d, const Par& par, double* U, size_t su, double* P, size_t sp, uint8_t* flags, double* atmo, cudaStream_t s);
cudaError_t launch_prim2con(const Dims& d, const Par& par, double* U, size_t su, double* P, size_t sp, cudaStream_t s);
cudaError_t launch_ccz4_algebra(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* K, size_t sk, cudaStream_t s);
cudaError_t launch_adv_ko(const Dims& d, const Par& par, const double* U, size_t su, double* K, size_t sk, const Fuse& fz, cudaStream_t s);
cudaError_t launch_point_flux(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* Wk, size_t sw, cudaStream_t s);
cudaError_t launch_recon(int dir, const Dims& d, const Par& par, const double* U, size_t su, const double* Wk, size_t sw, double* K, size_t sk, const Fuse& fz, cudaStream_t s);
cudaError_t launch_rk_combine(const Dims& d, int nfields, double* Uout, size_t so, const double* U0, size_t s0,
                              int nk, const double* const* K, const size_t* sk, const double* coef, double dt, cudaStream_t s);
cudaError_t launch_copy_fields(const Dims& d, int nfields, double* dst, size_t sd, const double* src, size_t ss, cudaStream_t s);
cudaError_t launch_count_flags(const Dims& d, const uint8_t* flags, unsigned long long* counts, cudaStream_t s);
double probe_fp64(cudaStream_t s);
cudaError_t launch_m1_point(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, const double* V, size_t sv,
                            double* Wk, size_t sw, cudaStream_t s);
cudaError_t launch_m1_div(const Dims& d, const Par& par, const double* U, size_t su, const double* V, size_t sv, const double* Wk, size_t sw,
                          double* KV, size_t sk, cudaStream_t s);
cudaError_t launch_m1_implicit(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* V, size_t sv,
                               double* R, size_t sr, double adt, uint8_t* flags, cudaStream_t s);
cudaError_t launch_m1_gravity(const Dims& d, const Par& par, const double* U, size_t su, const double* V, size_t sv, const double* Wk, size_t sw,
                              double* K, size_t sk, cudaStream_t s);
cudaError_t launch_les(const Dims& d, const Par& par, const double* U, size_t su, const double* P, size_t sp, double* A, size_t sa,
                       double* Wk, size_t sw, cudaStream_t s);
cudaError_t launch_prolong(const Dims& dc, const double* Uc, size_t sc, const Dims& df, double* Uf, size_t sf, int nfields,
                           const int origin[3], const int lo[3], const int hi[3], cudaStream_t s);
cudaError_t launch_restrict(const Dims& df, const double* Uf, size_t sf, const Dims& dc, double* Uc, size_t sc, int nfields, const int origin[3], cudaStream_t s);
cudaError_t launch_dense(const Dims& d, int nfields, double* Uout, size_t so, const double* U0, size_t s0, int nk, const double* const* K,
                         const size_t* sk, const double* c, int with_u0, cudaStream_t s);
cudaError_t launch_m1_backreact(const Dims& d, const Par& par, const double* R, size_t sr, double* K, size_t sk, cudaStream_t s);
}  // namespace mhd
