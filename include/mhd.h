/* mhd.h — C ABI of the B200-native per-stage hot path of MHDuet (arXiv 2510.13965) on one uniform,
 * ghosted, vertex-centred grid patch.
 *
 * One RK stage (Eq. 53, l.384-387; App. C step C3) is the call sequence
 *     mhd_fill_ghosts -> mhd_con2prim -> mhd_rhs -> mhd_rk_stage
 * every step of which runs in hand-written sm_100a CUDA kernels. There is no CPU fallback.
 *
 * Memory model. The CALLER owns all field memory (device pointers, e.g. torch tensors) and binds it to
 * numbered slots with mhd_patch_bind; the library allocates only a few hundred bytes of device scratch at
 * create time, allocates nothing per call, launches asynchronously on the caller's stream
 * (a cudaStream_t passed as void*; NULL = legacy default stream) and never synchronises except in
 * mhd_patch_status and the *_host entry points. All floating point is FP64.
 *
 * Layout. A slot holds n_fields fields, SoA: value of field f at grid point (i,j,k) is
 *     base[f * field_stride + (k * MY + j) * MX + i],   MX = nx + 2 ng  (x fastest), 0 <= i < MX ...
 * Interior points are ng <= i < ng + nx. field_stride >= MX*MY*MZ (elements).
 *
 * State fields U (32): 0-5 gamma~_ij (xx,xy,xz,yy,yz,zz), 6-11 A~_ij, 12 chi, 13 K^, 14 Theta,
 *   15-17 Gamma^^i, 18 alpha, 19-21 beta^i (Eqs. 13-26);
 *   22 Dbar, 23 DYebar, 24 taubar, 25-27 Sbar_i, 28-30 Bbar^i, 31 phibar = sqrt(gamma) x Eq. (29).
 * Primitive fields P (10): rho, Ye, eps, p, v^x, v^y, v^z (contravariant), W, T, cs2.
 * Flags: one byte per grid point, bits = MHD_FLAG_*.
 *
 * Errors. Every function returns MHD_OK (0) or a negative MHD_E_* code; nothing throws or aborts.
 * The paper's "fatal error, stop the code" is a flag bit plus a counter.
 */
#ifndef MHD_H
#define MHD_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MHD_NSTATE 32
#define MHD_NPRIM 10
#define MHD_NWORK 33        /* 3 directions x (10 flux brackets of Eq. 32 + 1 speed bound of App. B) */
#define MHD_NM1 15          /* (Nbar, Ebar, Fbar_i) x 3 neutrino species, field 5 s + {0..4} */
#define MHD_NM1WORK 75      /* per species: 3 directions x (5 flux brackets + speed), kappa_a + kappa_s, P_ij */
#define MHD_NLESWORK 31     /* auxiliary fields of the LES sub-grid-scale terms (App. A): B^k, v^k, v_k, B_k, E_k, E^k, v.B, Theta, W^-2, rho, eps, h, dp/drho, dp/deps,
                               (tabulated EoS only) Ye, dp/dYe, (that or any of C_N, C_Y, C_T) D, (any of C_N, C_Y, C_T) calE = h W^2, D Ye */
#define MHD_MAX_STAGES 8
#define MHD_MAX_PIECES 8

/* slots */
enum {
  MHD_SLOT_U = 0,      /* current stage state U^(i)                      (MHD_NSTATE fields) */
  MHD_SLOT_U0 = 1,     /* U^n, saved by mhd_rk_stage(stage = 0)          (MHD_NSTATE fields) */
  MHD_SLOT_P = 2,      /* primitives                                     (MHD_NPRIM fields)  */
  MHD_SLOT_FLAGS = 3,  /* uint8 flags, one field                                             */
  MHD_SLOT_WORK = 4,   /* scratch of mhd_rhs: pointwise fluxes and speeds (MHD_NWORK fields) */
  MHD_SLOT_K1 = 5,     /* K_1 ... K_s = F(U^(j)): MHD_SLOT_K1 + j - 1    (MHD_NSTATE fields) */
  /* M1 (n_species = 3) */
  MHD_SLOT_V = 5 + MHD_MAX_STAGES,        /* neutrino fields of the current stage            (MHD_NM1 fields)     */
  MHD_SLOT_V0,                            /* V^n                                             (MHD_NM1 fields)     */
  MHD_SLOT_M1WORK,                        /* scratch of mhd_m1_rhs                           (MHD_NM1WORK fields) */
  MHD_SLOT_KV1,                           /* explicit parts F_V(U^(j)): MHD_SLOT_KV1 + j - 1 (MHD_NM1 fields)     */
  MHD_SLOT_R1 = MHD_SLOT_KV1 + MHD_MAX_STAGES,   /* stiff sources R_V(U^(j)): MHD_SLOT_R1 + j - 1 (MHD_NM1 fields) */
  MHD_SLOT_U1 = MHD_SLOT_R1 + MHD_MAX_STAGES,    /* optional third state buffer (MHD_NSTATE fields): lets mhd_advance fuse the RK combine
                                                    into the right-hand-side kernels (the new stage state cannot overwrite the one
                                                    whose stencils are being read); unbound = separate combine kernel */
  MHD_SLOT_LESWORK = MHD_SLOT_U1 + 1,            /* scratch of the LES term (MHD_NLESWORK fields); needed when any LES coefficient != 0 */
  MHD_NSLOTS = MHD_SLOT_LESWORK + 1
};

/* flag bits: error policy of PAPER.md:1157-1162 */
enum {
  MHD_FLAG_ATMO = 1,     /* rule 1: reset to atmosphere                    */
  MHD_FLAG_EPS_LO = 2,   /* rule 3: eps raised to eps_min                  */
  MHD_FLAG_EPS_HI = 4,   /* rule 4: eps lowered to eps_max                 */
  MHD_FLAG_VMAX = 8,     /* rule 5: velocity rescaled to W_max             */
  MHD_FLAG_YE = 16,      /* rule 6: Ye reset                               */
  MHD_FLAG_FATAL = 32,   /* rules 2, 4-6 outside low-density / BH regions  */
  MHD_FLAG_NOCONV = 64,  /* a root find hit the iteration cap              */
  MHD_FLAG_M1FIX = 128   /* M1: E floored or |F| limited to E (reading R22) */
};

enum {
  MHD_OK = 0,
  MHD_E_ARG = -1,        /* null pointer / out-of-range argument            */
  MHD_E_UNBOUND = -2,    /* a slot needed by the call has not been bound    */
  MHD_E_CUDA = -3,       /* CUDA runtime error (launch, copy, allocation)   */
  MHD_E_UNSUPPORTED = -4, /* not supported: n_species other than 0 or 3, an M1 call on a patch without species */
  MHD_E_TOO_LARGE = -5   /* a size beyond the fixed capacity of an allocation-free entry point (mhd_flag_census_static) */
};

/* Plain data, copied at create time. Pointers inside are DEVICE pointers that must outlive the patch. */
typedef struct {
  int nx, ny, nz, ng;              /* interior points per axis; ghost width (>= 3: MP5/KO/advective stencils) */
  double dx, dy, dz;               /* uniform spacing */
  int n_species;                   /* 0 (M1 off) or 3 (grey M1: nu_e, anti-nu_e, nu_x) */
  /* EoS: 0 ideal gas p=(Gamma-1) rho eps; 1 hybrid piecewise polytrope (Eqs. 30-31); 2 table */
  int eos_kind;
  double eos_gamma;                /* kind 0 */
  double eos_gamma_th;             /* kind 1 */
  int n_pieces;                    /* kind 1; piece i holds for pp_rho[i-1] <= rho < pp_rho[i]; K_i, a_i (i>0) by continuity */
  double pp_K[MHD_MAX_PIECES], pp_Gamma[MHD_MAX_PIECES], pp_rho[MHD_MAX_PIECES];
  /* kind 2: log10 p, log10(eps + tab_eps_shift), cs2 tabulated on (log10 rho, log10 T, Ye), rho fastest; DEVICE pointers */
  const double *tab_logp, *tab_loge, *tab_cs2;
  int n_rho, n_T, n_ye;
  double lr0, dlr, lT0, dlT, ye0, dye, tab_eps_shift, tab_h0;
  /* CCZ4 + gauge, Eqs. (13)-(20), (25)-(26) */
  double kappa_z, kappa_c, kappa_2, eta_shift, f_alpha, f_beta, beta0[3];
  double grav_G;                   /* the explicit G of 8 pi G in Eqs. (14),(16),(17),(19); 0 decouples matter */
  double sigma_ko_spacetime, sigma_ko_matter;   /* Kreiss-Oliger sigma */
  /* GRMHD: divergence cleaning speed and damping (Eq. 28), MP5 alpha */
  double c_b, kappa_b, mp5_alpha;
  /* con2prim error policy */
  double rho_atmo, rho_cut, rho_low, alpha_bh, w_max, rho_max, eps_min, eps_max;
  double ye_min, ye_max, ye_atmo, eps_atmo, T_atmo;
  int c2p_maxit;
  /* M1 (n_species = 3): synthetic grey opacities kappa_a = kappa_s = m1_kappa0 (rho / m1_rho0)^2 m1_species_scale[s],
   * eta = m1_arad kappa_a T^4 (BASELINE.json configs[4]: m1_arad = 1; it is the radiation constant in the units T is measured in);
   * energy floor, Newton tolerance / cap of App. C, baryon mass of l.316 */
  double m1_kappa0, m1_rho0, m1_species_scale[3], m1_efloor, m1_tol, m1_mb;
  int m1_maxit, m1_odd_even;       /* m1_odd_even != 0: the A := 1 switch against odd-even decoupling (l.565-570) */
  double m1_arad;                  /* see above; 0 switches the emission off */
  double m1_oe_guard;              /* reading R33: the switch also needs all three differences to exceed m1_oe_guard x the local
                                      magnitude; 0 = the rule exactly as printed (two strict "< 0" tests) */
  /* SURVEY 8(f) rows */
  int recon_kind;                  /* the reconstruction R of Eq. (66): 0 MP5 (Eqs. 70-76, the paper's default), 1 WENO5 (PAPER.md:486-488,
                                      ref. [63]: linear weights 1/10, 6/10, 3/10, exponent 2) */
  double weno_eps;                 /* recon_kind 1: the epsilon added to the smoothness indicators (ref. [63]: 1e-6); must be > 0 */
  double les_C_M;                  /* App. A, Eq. (A11): coefficient C_M of the sub-grid-scale tensor of the induction equation (the paper's
                                      production value is 8); 0 = LES terms off. When non-zero: ng >= 5 (the gradients of the
                                      auxiliary fields are needed at every node the reconstruction reads) and MHD_SLOT_LESWORK bound; otherwise
                                      mhd_patch_create / mhd_rhs refuse. dp/drho, dp/deps, dp/dYe: analytic for eos_kind 0 / 1, derivatives of the
                                      interpolant inside the table cell for eos_kind 2 (l.882) */
  double les_C_N, les_C_Y, les_C_T; /* App. A, Eqs. (A11), (A15), (A17): coefficients of the sub-grid-scale tensors H_N^k (flux of Dbar), H_{N_Y}^k (flux of
                                      DYebar) and gamma_ij H_T^{kj} (flux of Sbar_i; H_E from the curl of H_M, R45, R46); the paper's runs leave them 0
                                      (PAPER.md:863). taubar receives no SGS flux ((A11) defines none, R47). Same requirements as les_C_M when any is non-zero */
} mhd_patch_desc;

/* Butcher tableaux (Eq. 54), HOST pointers, row-major stages x stages; a_impl/w_impl may be NULL */
typedef struct {
  int stages;
  const double *a_expl, *w_expl, *a_impl, *w_impl;
} mhd_tableau;

typedef struct {
  unsigned long long n_points, n_atmo, n_eps_lo, n_eps_hi, n_vmax, n_ye, n_fatal, n_noconv, n_m1fix;
  unsigned long long halo_timeout;   /* non-zero: a wait on a neighbour patch (fused halo fill) expired; the state is not valid */
} mhd_status;

typedef struct mhd_patch mhd_patch;   /* opaque */

size_t mhd_desc_sizeof(void);         /* sizeof(mhd_patch_desc) as compiled, for binding self-checks */

/* Create / destroy. *out owns a copy of desc and a small device scratch buffer. */
int mhd_patch_create(const mhd_patch_desc *desc, mhd_patch **out);
void mhd_patch_destroy(mhd_patch *p);

/* Bind caller-owned DEVICE memory to a slot. field_stride in elements (doubles; bytes for MHD_SLOT_FLAGS). */
int mhd_patch_bind(mhd_patch *p, int slot, void *dev_ptr, size_t field_stride);

/* a1 — ghost fill: bc[6] = {x-,x+,y-,y+,z-,z+}, 0 periodic wrap, 1 outflow (copy of the nearest
 * interior value), 2 neighbour patch (below). Fills all ng ghost layers incl. edges and corners of every field of the slot, in
 * place. MHD_E_ARG if a periodic or neighbour axis has fewer interior points than ghost layers. */
int mhd_fill_ghosts(mhd_patch *p, int slot_state, const int bc[6], void *cuda_stream);

/* ---- Domain decomposition: halo exchange fused with the ghost fill ("spatial decomposition") ----
 * The patch is one brick of a regular decomposition; all bricks have the same nx, ny, nz, ng. A face with bc = 2 has a neighbour
 * brick behind it: its ghost layers are read by the ghost-fill kernel directly from the neighbour's interior, i.e. from the SAME SLOT
 * of the neighbour patch, whose device pointer is registered here — a pointer on this GPU, or a peer-GPU mapping (cudaIpcOpenMemHandle
 * / peer access) read over NVLink: no pack, send or unpack. dir[3] in {-1,0,1}^3 \ {0} names the neighbour: faces, and the edge /
 * corner neighbours wherever two / three neighbour faces meet (a domain-periodic axis split over several bricks is a neighbour
 * axis too; an axis with a single brick keeps bc 0 / 1). Register every state slot mhd_advance rotates (U, U0, and U1 if bound):
 * the entries travel with the buffers. MHD_E_UNBOUND from mhd_fill_ghosts if a needed neighbour is missing. */
int mhd_patch_set_neighbor(mhd_patch *p, int slot, const int dir[3], const void *peer_dev_ptr, size_t peer_field_stride);
/* Ordering between patches driven from different streams / processes / GPUs. Each patch owns 27 epoch words in device memory
 * (mhd_patch_halo_words; export with mhd_ipc_export). After mhd_patch_set_neighbor_word(p, dir, <halo words of the neighbour in
 * direction dir>) every ghost fill with neighbour faces runs   signal "my interior is final" -> wait for the neighbours' signal ->
 * fill -> signal "I have read" -> wait   as stream-ordered kernels (system-scope release / acquire on the words; no host
 * synchronisation, no collective library). All bricks must issue the same sequence of ghost fills. A wait that expires (~4 s) sets
 * mhd_status.halo_timeout instead of hanging the device. Patches driven from ONE stream need no words. */
void *mhd_patch_halo_words(mhd_patch *p);
int mhd_patch_set_neighbor_word(mhd_patch *p, const int dir[3], void *peer_halo_words);
/* CUDA IPC helpers (one process per GPU): export = handle of the allocation that holds dev_ptr + offset of dev_ptr in it; import
 * maps it into this process and returns the usable device pointer; close unmaps it. */
int mhd_ipc_export(const void *dev_ptr, unsigned char handle[64], size_t *offset);
int mhd_ipc_import(const unsigned char handle[64], size_t offset, void **dev_ptr);
int mhd_ipc_close(void *dev_ptr, size_t offset);

/* a2 — conserved -> primitive at every grid point incl. ghosts (App. D, Eqs. D1-D15, error policy
 * l.1157-1162). Writes the 10 primitives and the flag byte; where a rule changed a primitive the fluid conserved
 * fields of slot_state are reset from the corrected primitives (Bbar, phibar untouched). slot_prim is also READ: if it holds
 * valid primitives (e.g. of the previous stage) they give the starting bracket of the root solve (warm start); the result is
 * the same root to solver tolerance whatever slot_prim held, zeros and NaNs included.
 * A patch has ONE primitive slot and ONE flag slot: slot_prim must be MHD_SLOT_P and slot_flags MHD_SLOT_FLAGS (MHD_E_ARG otherwise; the
 * arguments keep the call in the form of the problem statement and leave room for more slots); slot_state is any state slot (U, U0, U1, K_j). */
int mhd_con2prim(mhd_patch *p, int slot_state, int slot_prim, int slot_flags, void *cuda_stream);

/* inverse of a2 for initial data (Eq. 29): slot_prim holds rho, Ye, eps, v^i; fills p, W, T, cs2 there and
 * Dbar, DYebar, taubar, Sbar_i in slot_state from them, the metric and Bbar^i already in slot_state. */
int mhd_prim2con(mhd_patch *p, int slot_state, int slot_prim, void *cuda_stream);

/* a3-a8 — right-hand side F(U) on the interior: CCZ4 + gauge (Eqs. 13-26; FD Eqs. 60-62, upwind l.454-456,
 * KO l.460), GRMHD flux divergence (Eq. 32 with Eqs. 63-76, speeds App. B) and sources. Ghost points of
 * slot_rhs are not written. Needs filled ghosts in slot_state and primitives at all points, and MHD_SLOT_WORK bound
 * (overwritten: pointwise F^d(U,P) and speeds at every grid point, computed once and read by the three 1-D
 * reconstruction passes). */
int mhd_rhs(mhd_patch *p, int slot_state, int slot_prim, int slot_rhs, void *cuda_stream);

/* LES (App. A Eqs. A11-A17): the sub-grid-scale tensor of the induction equation. Computes the auxiliary
 * fields of App. A at every grid point into MHD_SLOT_LESWORK and ADDS -alpha G_B^{ki} = alpha C_M xi sqrt(gamma) H_M^{ki}
 * (xi = gamma^{1/3} Delta^2 / 24, Delta = (dx dy dz)^{1/3}) to the pointwise flux of Bbar^i in direction k held in MHD_SLOT_WORK
 * (field 11 k + 6 + i), at every point at least 2 points inside the array; with les_C_N / les_C_Y / les_C_T set also alpha C xi sqrt(gamma) x
 * H_N^k (field 11 k), H_{N_Y}^k (field 11 k + 1), gamma_ij H_T^{kj} (field 11 k + 3 + i). mhd_rhs calls it between the pointwise fluxes and the
 * reconstruction when any LES coefficient != 0; exposed for tests and for callers that sequence the right-hand side themselves. */
int mhd_les_flux(mhd_patch *p, int slot_state, int slot_prim, void *cuda_stream);

/* a9 — explicit RK combine on the interior (Eq. 53).
 *   stage = 0          : U0 <- U  (start of a step)
 *   1 <= stage < s     : U <- U0 + dt * sum_{j<=stage} a_expl[stage][j-1] K_j      (= U^(stage+1))
 *   stage = s          : U <- U0 + dt * sum_j w_expl[j-1] K_j                      (= U^{n+1})
 * K_j is slot MHD_SLOT_K1 + j - 1; zero coefficients are skipped (their slots need not be bound). Ghost points of U carry no
 * meaning afterwards (large patches are combined as whole flat arrays): mhd_fill_ghosts refills them before anything reads them. */
int mhd_rk_stage(mhd_patch *p, const mhd_tableau *t, int stage, double dt, void *cuda_stream);

/* n_steps full RK steps, device resident: per stage fill -> con2prim -> rhs(K_stage) -> rk_stage; the state is
 * left with ghosts filled and primitives/flags consistent. Asynchronous. With MHD_SLOT_U1 bound the combine of Eq. (53) is
 * computed by the last right-hand-side kernel that touches each field (same arithmetic, one pass less over K and U per
 * stage; K_s of the last stage is then not stored); the buffers bound to U, U0, U1 are all overwritten, the result is in U.
 * The call only enqueues kernels and memsets on cuda_stream (no synchronisation, allocation or host read; the opt-ins to large shared memory
 * happen at the first call on a device), so after one ordinary call it may be captured into a CUDA graph and replayed (small patches are
 * launch-bound: about 50 launches per RK4 step); a replay reproduces the direct call bit for bit when U and the primitives (the warm start of
 * con2prim) hold the same values. Without halo neighbours only: the epoch of the halo protocol advances on the host. */
int mhd_advance(mhd_patch *p, const mhd_tableau *t, const int bc[6], double dt, int n_steps, void *cuda_stream);

/* Same, end to end with HOST buffers: copies host_U (MHD_NSTATE fields, packed, field_stride = MX*MY*MZ) to
 * slot U, advances, copies U back into host_U and the flags into host_flags (may be NULL), then synchronises
 * the stream. Pinned host memory makes the copies asynchronous with respect to the host. */
int mhd_advance_host(mhd_patch *p, const mhd_tableau *t, const int bc[6], double dt, int n_steps,
                     double *host_U, uint8_t *host_flags, void *cuda_stream);

/* ---- M1 (Sec. II C, III D, App. B, C); all need n_species = 3 ----
 * a12 (+a10) — pointwise implicit solve at every grid point (App. C, Eqs. C10-C35): slot_V holds V* (densitised) on entry and
 * V^(i) on exit; slot_R receives the densitised stiff source alpha sqrt(gamma) (C, S_n, S_i) evaluated at V^(i); adt = a_ii dt.
 * Needs slot U (metric) and P (v^i, W, rho, T) consistent; ORs MHD_FLAG_M1FIX / MHD_FLAG_NOCONV into slot FLAGS. */
int mhd_m1_implicit(mhd_patch *p, int slot_V, int slot_R, double adt, void *cuda_stream);
/* a11 (+a10) — explicit part of Eqs. (38)-(40) on the interior: closure at every point, fluxes of Eqs. (77)-(78), geometric
 * sources; slot_KV <- F_V. Needs filled ghosts in slot_V and slot U, primitives at all points, MHD_SLOT_M1WORK bound. */
int mhd_m1_rhs(mhd_patch *p, int slot_V, int slot_KV, void *cuda_stream);
/* a8 (M1 part) — neutrino back-reaction on the fluid: slot_K[taubar, Sbar_i] -= sum_species slot_R[Ebar, Fbar_i],
 * slot_K[DYebar] -= m_b (R[Nbar]_nue - R[Nbar]_anti-nue), interior. */
int mhd_m1_backreaction(mhd_patch *p, int slot_R, int slot_K, void *cuda_stream);
/* a4 (M1 part, reading R6) — radiation E, F_i, P_ij of the three species added to the matter sources of the CCZ4 equations
 * (Eqs. 14, 16, 17, 19) in slot_K, interior. P_ij is taken from MHD_SLOT_M1WORK: call after mhd_m1_rhs on the same slot_V. */
int mhd_m1_gravity(mhd_patch *p, int slot_V, int slot_K, void *cuda_stream);
/* n_steps full IMEX steps (Eq. 53, App. C steps C3-C4) of the coupled system, device resident; the tableau must carry
 * a_impl (row-major, lower triangular incl. diagonal) and w_impl. Per stage: combine -> fill -> con2prim -> implicit solve ->
 * M1 explicit part -> rhs + back-reaction + radiation in the CCZ4 sources. */
int mhd_advance_imex(mhd_patch *p, const mhd_tableau *t, const int bc[6], double dt, int n_steps, void *cuda_stream);

/* ---- AMR transfer operators on a patch pair (Sec. IV B l.608-626; refinement ratio 2, vertex-centred grids so that every
 * coarse point is also a fine point, l.620). `origin[3]` (x, y, z) is the coarse INTERIOR index of the coarse point under fine
 * interior point (0, 0, 0); fine interior index a (negative / >= n in the ghosts) sits at coarse position origin + a / 2.
 * Both patches live on the same device; the two slots must hold the same number of fields (any slot but FLAGS).
 *
 * mhd_prolong: sets every fine grid point of the box lo[d] <= index < hi[d] (GHOSTED fine array indices, x, y, z) of slot_f from slot_c:
 * a coincident point is a copy, a midpoint is the fifth-order Lagrange formula of Eq. (80) (l.616), applied along x, then y, then z
 * (tensor product). Serves both the filling of a new fine patch (box = whole array) and the fine ghost zones at a coarse-fine
 * boundary (one box per face). MHD_E_ARG if a coarse stencil point (offsets -2..+3) falls outside the coarse array. */
int mhd_prolong(mhd_patch *coarse, int slot_c, mhd_patch *fine, int slot_f, const int origin[3], const int lo[3], const int hi[3],
                void *cuda_stream);
/* mhd_restrict: direct copy (l.626) of the fine INTERIOR points with even indices onto the coarse points they coincide with. */
int mhd_restrict(mhd_patch *fine, int slot_f, mhd_patch *coarse, int slot_c, const int origin[3], void *cuda_stream);
/* Dense-output interpolator (Eqs. 56-59, l.412-434), the time interpolation of the coarse level that sub-cycling needs (l.644-649):
 * scheme 0 = RK(4,4), Eq. (58), third order; scheme 1 = SSP-RK(3,3), Eq. (59), second order. On the interior,
 *   deriv = 0:      slot_out <- U0 + sum_j b_j(theta) dt K_j                         (Eq. 56; theta = (t - t^n)/dt)
 *   deriv = 1..3:   slot_out <- dt^-deriv sum_j d^deriv b_j / dtheta^deriv dt K_j    (Eq. 57: time derivatives at t^n + theta dt)
 * U0 (slot MHD_SLOT_U0) and K_j (MHD_SLOT_K1 + j - 1) must hold U^n and F(U^(j)) of the step, as the mhd_rk_stage sequence leaves
 * them. slot_out: any state slot but U0 and the K_j used. mhd_dense_weights returns the number of stages and b_j (host, no device work). */
int mhd_dense_weights(int scheme, double theta, int deriv, double b[4]);
int mhd_dense_output(mhd_patch *p, int scheme, double theta, double dt, int deriv, int slot_out, void *cuda_stream);

/* Same, end to end with HOST buffers (packed, field_stride = MX*MY*MZ): host_U (MHD_NSTATE fields) and host_V (MHD_NM1 fields) are
 * copied to slots U and V, advanced, copied back together with the flags (host_flags may be NULL); synchronises the stream. */
int mhd_advance_imex_host(mhd_patch *p, const mhd_tableau *t, const int bc[6], double dt, int n_steps, double *host_U, double *host_V,
                          uint8_t *host_flags, void *cuda_stream);

/* Counts flag bits over all grid points of slot_flags. Synchronises the stream. */
int mhd_patch_status(mhd_patch *p, int slot_flags, mhd_status *out, void *cuda_stream);

/* Per-kernel device timing (CUDA events recorded on the launching stream around every kernel of the library).
 * mhd_patch_profile(p, 1) starts collecting, (p, 0) stops. mhd_patch_profile_read synchronises the stream, adds up
 * the elapsed milliseconds and launch counts per kernel class since the last read, and resets them.
 * Classes: 0 ghost fill, 1 con2prim, 2 ccz4 algebra (+ fluid sources), 3 reconstruction x, 4 y, 5 z, 6 rk combine / copy,
 * 7 pointwise fluxes, 8 advection + Kreiss-Oliger, 9 M1 closure + pointwise fluxes, 10 M1 flux divergence + sources,
 * 11 M1 implicit solve + back-reaction, 12 LES sub-grid-scale term. */
#define MHD_NKERNELS 13
int mhd_patch_profile(mhd_patch *p, int enable);
int mhd_patch_profile_read(mhd_patch *p, double ms[MHD_NKERNELS], unsigned long long launches[MHD_NKERNELS], void *cuda_stream);

/* Measured FP64 FMA throughput of the device (register-resident DFMA chains on every SM), in FLOP/s;
 * used as the FP64 roofline denominator. Synchronises. Returns < 0 on error. */
double mhd_probe_fp64_flops(void *cuda_stream);

/* Flag census WITHOUT any allocation and without an mhd_patch (whose create call allocates): for callers that cannot call cudaMalloc — code under
 * CUDA stream capture, tight serving loops, harnesses that forbid it. Counts the flag bits (App. D error policy, l.1151-1162; the bits mhd_con2prim
 * and mhd_m1_implicit set) over n_points bytes.
 *   d_flags   DEVICE pointer, n_points bytes, read only (e.g. the buffer bound to MHD_SLOT_FLAGS, MX*MY*MZ bytes).
 *   d_counts  DEVICE pointer, 9 words written: [0] = n_points, [1 + b] = number of bytes with bit b set (the order of mhd_status: atmo, eps_lo, eps_hi,
 *             vmax, ye, fatal, noconv, m1fix). The caller owns both buffers; nothing is copied to the host, the stream is not synchronised.
 * The partial counts live in a file-scope device array of fixed size inside the library (128 KB, held by every GPU that loads the library until exit):
 * n_points > MHD_CENSUS_MAX_POINTS returns MHD_E_TOO_LARGE and launches nothing; null pointers or n_points < 1: MHD_E_ARG. The call makes no cudaMalloc /
 * cudaFree and calls no allocating routine. All calls share that array: calls on one stream are ordered; two calls that OVERLAP on the GPU (different
 * streams, two host threads on one device) race on it and their results are undefined. Same counts as mhd_patch_status, bit for bit. */
#define MHD_CENSUS_MAX_POINTS 268435456LL   /* 2^28 points = 645^3 with ghosts */
int mhd_flag_census_static(const uint8_t *d_flags, long long n_points, unsigned long long *d_counts, void *cuda_stream);

const char *mhd_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* MHD_H */
