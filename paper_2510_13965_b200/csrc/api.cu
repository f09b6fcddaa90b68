// C ABI of libmhd_b200 (see include/mhd.h): argument checking, slot bookkeeping and kernel sequencing only.
#include <math.h>
#include <new>
#include <string.h>
#include "mhd_internal.cuh"

using namespace mhd;

namespace {

int slot_fields(int slot) {
  if (slot == MHD_SLOT_P) return MHD_NPRIM;
  if (slot == MHD_SLOT_FLAGS) return 1;
  if (slot == MHD_SLOT_WORK) return MHD_NWORK;
  if (slot == MHD_SLOT_M1WORK) return MHD_NM1WORK;
  if (slot == MHD_SLOT_LESWORK) return MHD_NLESWORK;
  if (slot >= MHD_SLOT_V) return MHD_NM1;
  return MHD_NSTATE;
}
bool slot_ok(const mhd_patch* p, int slot) { return slot >= 0 && slot < MHD_NSLOTS && p->slot[slot].ptr != nullptr; }
bool is_state_slot(int slot) { return slot == MHD_SLOT_U || slot == MHD_SLOT_U0 || slot == MHD_SLOT_U1 || (slot >= MHD_SLOT_K1 && slot < MHD_SLOT_K1 + MHD_MAX_STAGES); }
bool is_m1_slot(int slot) { return slot >= MHD_SLOT_V && slot < MHD_SLOT_U1 && slot != MHD_SLOT_M1WORK; }
int les_impl(mhd_patch* p, int slot_state, int slot_prim, cudaStream_t s);
bool les_on(const Par& q) { return q.les_C_M != 0.0 || q.les_C_N != 0.0 || q.les_C_Y != 0.0 || q.les_C_T != 0.0; }
double* dptr(const mhd_patch* p, int slot) { return (double*)p->slot[slot].ptr; }

// piecewise-polytrope continuity constants: K_i, a_i for i > 0
void finish_eos(Par& q) {
  q.pp_a[0] = 0.0;
  for (int i = 1; i < q.n_pieces; ++i) {
    const double rb = q.pp_rho[i - 1];
    q.pp_K[i] = q.pp_K[i - 1] * pow(rb, q.pp_Gamma[i - 1] - q.pp_Gamma[i]);
    const double em = q.pp_a[i - 1] + q.pp_K[i - 1] / (q.pp_Gamma[i - 1] - 1.0) * pow(rb, q.pp_Gamma[i - 1] - 1.0);
    q.pp_a[i] = em - q.pp_K[i] / (q.pp_Gamma[i] - 1.0) * pow(rb, q.pp_Gamma[i] - 1.0);
  }
}

// RAII event pair around one kernel launch when profiling is on
struct Timed {
  mhd_patch* p; cudaStream_t s; mhd_patch::Ev ev; bool on;
  Timed(mhd_patch* p_, int cls, cudaStream_t s_) : p(p_), s(s_), on(p_->profiling) {
    if (!on) return;
    if (!p->pool.empty()) { ev = p->pool.back(); p->pool.pop_back(); }
    else { cudaEventCreate(&ev.a); cudaEventCreate(&ev.b); }
    ev.cls = cls;
    cudaEventRecord(ev.a, s);
  }
  ~Timed() {
    if (!on) return;
    cudaEventRecord(ev.b, s);
    p->events.push_back(ev);
  }
};

// a3-a8: the kernels of one right-hand-side evaluation; fz (optional) fuses the RK combine into the last kernel that touches each field
int rhs_impl(mhd_patch* p, int slot_state, int slot_prim, int slot_rhs, const Fuse& fz, cudaStream_t s) {
  double* Wk = dptr(p, MHD_SLOT_WORK);
  const size_t sw = p->slot[MHD_SLOT_WORK].stride;
  const double* U = dptr(p, slot_state);
  const double* P = dptr(p, slot_prim);
  double* K = dptr(p, slot_rhs);
  const size_t su = p->slot[slot_state].stride, sp = p->slot[slot_prim].stride, sk = p->slot[slot_rhs].stride;
  { Timed tm(p, 2, s); if (launch_ccz4_algebra(p->dims, p->par, U, su, P, sp, K, sk, s) != cudaSuccess) return MHD_E_CUDA; }
  { Timed tm(p, 8, s); if (launch_adv_ko(p->dims, p->par, U, su, K, sk, fz, s) != cudaSuccess) return MHD_E_CUDA; }
  { Timed tm(p, 7, s); if (launch_point_flux(p->dims, p->par, U, su, P, sp, Wk, sw, s) != cudaSuccess) return MHD_E_CUDA; }
  if (les_on(p->par)) { const int rc = les_impl(p, slot_state, slot_prim, s); if (rc != MHD_OK) return rc; }
  for (int dir = 0; dir < 3; ++dir) {
    Timed tm(p, 3 + dir, s);
    if (launch_recon(dir, p->dims, p->par, U, su, Wk, sw, K, sk, fz, s) != cudaSuccess) return MHD_E_CUDA;
  }
  return MHD_OK;
}


int les_impl(mhd_patch* p, int slot_state, int slot_prim, cudaStream_t s) {
  if (!slot_ok(p, MHD_SLOT_LESWORK) || !slot_ok(p, MHD_SLOT_WORK)) return MHD_E_UNBOUND;
  Timed tm(p, 12, s);
  return launch_les(p->dims, p->par, dptr(p, slot_state), p->slot[slot_state].stride, dptr(p, slot_prim), p->slot[slot_prim].stride,
                    dptr(p, MHD_SLOT_LESWORK), p->slot[MHD_SLOT_LESWORK].stride, dptr(p, MHD_SLOT_WORK), p->slot[MHD_SLOT_WORK].stride, s) == cudaSuccess
             ? MHD_OK : MHD_E_CUDA;
}

// n_steps full RK steps, the combine of Eq. (53) fused into the right-hand-side kernels (needs the third state buffer MHD_SLOT_U1).
// Three buffers rotate: one holds U^n for the whole step, each stage differentiates `cur` and writes the next stage state into the
// buffer that is neither `cur` nor U^n. Nothing is copied except, once per call, the result into the buffer bound to MHD_SLOT_U.
int stage_sequence_fused(mhd_patch* p, const mhd_tableau* t, const int bc[6], double dt, int n_steps, cudaStream_t s) {
  const Slot buf[3] = {p->slot[MHD_SLOT_U], p->slot[MHD_SLOT_U0], p->slot[MHD_SLOT_U1]};
  auto done = [&](int code) { p->slot[MHD_SLOT_U] = buf[0]; return code; };
  const int q = t->stages;
  for (int j = 0; j < q; ++j) if (!slot_ok(p, MHD_SLOT_K1 + j)) return MHD_E_UNBOUND;
  int rc, cur = 0;
  for (int step = 0; step < n_steps; ++step) {
    const int u0 = cur;                                      // U^n = the state entering the step, after the ghost fill and con2prim of stage 1 (R31)
    for (int st = 1; st <= q; ++st) {
      p->slot[MHD_SLOT_U] = buf[cur];
      if ((rc = mhd_fill_ghosts(p, MHD_SLOT_U, bc, s)) != MHD_OK) return done(rc);
      if ((rc = mhd_con2prim(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_FLAGS, s)) != MHD_OK) return done(rc);
      int w = 0;
      while (w == cur || w == u0) ++w;
      const double* coef = st < q ? t->a_expl + (size_t)st * q : t->w_expl;      // row of U^(st+1), or the weights
      Fuse fz;
      fz.Uout = (double*)buf[w].ptr; fz.so = buf[w].stride;
      fz.U0 = (const double*)buf[u0].ptr; fz.s0 = buf[u0].stride;
      fz.cself = dt * coef[st - 1];
      fz.write_k = st < q;                                   // K_q has no later reader
      for (int j = 0; j < st - 1; ++j)
        if (coef[j] != 0.0) { fz.Kp[fz.nk] = dptr(p, MHD_SLOT_K1 + j); fz.skp[fz.nk] = p->slot[MHD_SLOT_K1 + j].stride; fz.cp[fz.nk] = dt * coef[j]; ++fz.nk; }
      if ((rc = rhs_impl(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_K1 + st - 1, fz, s)) != MHD_OK) return done(rc);
      cur = w;
    }
  }
  if (cur != 0) {                                            // result lives in another buffer: copy it home (once per call)
    Timed tm(p, 6, s);
    if (launch_copy_fields(p->dims, MHD_NSTATE, (double*)buf[0].ptr, buf[0].stride, (const double*)buf[cur].ptr, buf[cur].stride, s) != cudaSuccess) return done(MHD_E_CUDA);
  }
  p->slot[MHD_SLOT_U] = buf[0];
  if ((rc = mhd_fill_ghosts(p, MHD_SLOT_U, bc, s)) != MHD_OK) return rc;
  return mhd_con2prim(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_FLAGS, s);
}

// n_steps full RK steps. "U0 <- U" at the start of a step is a swap of the two slot pointers, not a copy: the first
// combine of the step rewrites the whole interior of the new U buffer and the ghost fill that follows rewrites every
// ghost cell, so nothing of its old content survives. After an odd number of steps the result is copied back into the
// buffer the caller bound to MHD_SLOT_U (once per call, not once per step).
int stage_sequence(mhd_patch* p, const mhd_tableau* t, const int bc[6], double dt, int n_steps, cudaStream_t s) {
  int rc;
  if (!slot_ok(p, MHD_SLOT_U) || !slot_ok(p, MHD_SLOT_U0)) return MHD_E_UNBOUND;
  if (slot_ok(p, MHD_SLOT_U1) && slot_ok(p, MHD_SLOT_P) && slot_ok(p, MHD_SLOT_FLAGS) && slot_ok(p, MHD_SLOT_WORK) && n_steps > 0)
    return stage_sequence_fused(p, t, bc, dt, n_steps, s);
  bool swapped = false;
  auto swap_u = [&]() { Slot tmp = p->slot[MHD_SLOT_U]; p->slot[MHD_SLOT_U] = p->slot[MHD_SLOT_U0]; p->slot[MHD_SLOT_U0] = tmp; swapped = !swapped; };
  auto fail = [&](int code) { if (swapped) swap_u(); return code; };
  for (int step = 0; step < n_steps; ++step) {
    if ((rc = mhd_fill_ghosts(p, MHD_SLOT_U, bc, s)) != MHD_OK) return fail(rc);
    if ((rc = mhd_con2prim(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_FLAGS, s)) != MHD_OK) return fail(rc);
    // stage 1 reads U^n from the buffer that becomes U0
    if ((rc = mhd_rhs(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_K1, s)) != MHD_OK) return fail(rc);
    swap_u();
    if ((rc = mhd_rk_stage(p, t, 1, dt, s)) != MHD_OK) return fail(rc);
    for (int st = 2; st <= t->stages; ++st) {
      if ((rc = mhd_fill_ghosts(p, MHD_SLOT_U, bc, s)) != MHD_OK) return fail(rc);
      if ((rc = mhd_con2prim(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_FLAGS, s)) != MHD_OK) return fail(rc);
      if ((rc = mhd_rhs(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_K1 + st - 1, s)) != MHD_OK) return fail(rc);
      if ((rc = mhd_rk_stage(p, t, st, dt, s)) != MHD_OK) return fail(rc);
    }
  }
  if (swapped) {   // result lives in the caller's U0 buffer: copy it home and restore the binding
    Timed tm(p, 6, s);
    if (launch_copy_fields(p->dims, MHD_NSTATE, dptr(p, MHD_SLOT_U0), p->slot[MHD_SLOT_U0].stride, dptr(p, MHD_SLOT_U), p->slot[MHD_SLOT_U].stride, s) != cudaSuccess)
      return fail(MHD_E_CUDA);
    swap_u();
  }
  if ((rc = mhd_fill_ghosts(p, MHD_SLOT_U, bc, s)) != MHD_OK) return rc;
  return mhd_con2prim(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_FLAGS, s);
}

}  // namespace

extern "C" {

int mhd_advance_imex(mhd_patch* p, const mhd_tableau* t, const int bc[6], double dt, int n_steps, void* stream);

size_t mhd_desc_sizeof(void) { return sizeof(mhd_patch_desc); }

int mhd_patch_create(const mhd_patch_desc* desc, mhd_patch** out) {
  if (!desc || !out) return MHD_E_ARG;
  if (desc->nx < 1 || desc->ny < 1 || desc->nz < 1 || desc->ng < 3) return MHD_E_ARG;
  if (!(desc->dx > 0.0 && desc->dy > 0.0 && desc->dz > 0.0)) return MHD_E_ARG;
  if (desc->n_species != 0 && desc->n_species != 3) return MHD_E_UNSUPPORTED;
  if (desc->eos_kind < 0 || desc->eos_kind > 2) return MHD_E_ARG;
  if ((desc->les_C_M != 0.0 || desc->les_C_N != 0.0 || desc->les_C_Y != 0.0 || desc->les_C_T != 0.0) && desc->ng < 5) return MHD_E_UNSUPPORTED;
  if (desc->recon_kind < 0 || desc->recon_kind > 1 || (desc->recon_kind == 1 && !(desc->weno_eps > 0.0))) return MHD_E_ARG;
  if (desc->eos_kind == 1 && (desc->n_pieces < 1 || desc->n_pieces > MHD_MAX_PIECES)) return MHD_E_ARG;
  if (desc->eos_kind == 2 && (!desc->tab_logp || !desc->tab_loge || !desc->tab_cs2 || desc->n_rho < 2 || desc->n_T < 2 || desc->n_ye < 2 ||
                              !(desc->dlr > 0.0 && desc->dlT > 0.0 && desc->dye > 0.0))) return MHD_E_ARG;
  mhd_patch* p = new (std::nothrow) mhd_patch();
  if (!p) return MHD_E_ARG;
  p->desc = *desc;
  Dims& d = p->dims;
  d.nx = desc->nx; d.ny = desc->ny; d.nz = desc->nz; d.ng = desc->ng;
  d.mx = d.nx + 2 * d.ng; d.my = d.ny + 2 * d.ng; d.mz = d.nz + 2 * d.ng;
  d.sy = d.mx; d.sz = (long long)d.mx * d.my; d.npts = d.sz * d.mz;
  d.dx = desc->dx; d.dy = desc->dy; d.dz = desc->dz;
  Par& q = p->par;
  memset(&q, 0, sizeof(q));
  q.eos_kind = desc->eos_kind; q.n_pieces = desc->n_pieces; q.eos_gamma = desc->eos_gamma; q.eos_gamma_th = desc->eos_gamma_th;
  for (int i = 0; i < MHD_MAX_PIECES; ++i) { q.pp_K[i] = desc->pp_K[i]; q.pp_Gamma[i] = desc->pp_Gamma[i]; q.pp_rho[i] = desc->pp_rho[i]; }
  if (q.eos_kind == 1) finish_eos(q);
  q.tab_logp = desc->tab_logp; q.tab_loge = desc->tab_loge; q.tab_cs2 = desc->tab_cs2;
  q.n_rho = desc->n_rho; q.n_T = desc->n_T; q.n_ye = desc->n_ye;
  q.lr0 = desc->lr0; q.dlr = desc->dlr; q.lT0 = desc->lT0; q.dlT = desc->dlT; q.ye0 = desc->ye0; q.dye = desc->dye;
  q.tab_eps_shift = desc->tab_eps_shift; q.tab_h0 = desc->tab_h0;
  if (q.eos_kind == 2) {
    q.idlr = 1.0 / q.dlr; q.idlT = 1.0 / q.dlT; q.idye = 1.0 / q.dye;
    q.tab_rho_lo = pow(10.0, q.lr0); q.tab_rho_hi = pow(10.0, q.lr0 + q.dlr * (q.n_rho - 1));
  }
  q.kappa_z = desc->kappa_z; q.kappa_c = desc->kappa_c; q.kappa_2 = desc->kappa_2; q.eta_shift = desc->eta_shift;
  q.f_alpha = desc->f_alpha; q.f_beta = desc->f_beta; q.grav_G = desc->grav_G;
  for (int i = 0; i < 3; ++i) q.beta0[i] = desc->beta0[i];
  q.sigma_ko_spacetime = desc->sigma_ko_spacetime; q.sigma_ko_matter = desc->sigma_ko_matter;
  q.c_b = desc->c_b; q.kappa_b = desc->kappa_b; q.mp5_alpha = desc->mp5_alpha;
  q.rho_atmo = desc->rho_atmo; q.rho_cut = desc->rho_cut; q.rho_low = desc->rho_low; q.alpha_bh = desc->alpha_bh;
  q.w_max = desc->w_max; q.rho_max = desc->rho_max; q.eps_min = desc->eps_min; q.eps_max = desc->eps_max;
  q.ye_min = desc->ye_min; q.ye_max = desc->ye_max; q.ye_atmo = desc->ye_atmo; q.eps_atmo = desc->eps_atmo; q.T_atmo = desc->T_atmo;
  q.c2p_maxit = desc->c2p_maxit > 0 ? desc->c2p_maxit : 100;
  q.m1_kappa0 = desc->m1_kappa0; q.m1_rho0 = desc->m1_rho0 > 0.0 ? desc->m1_rho0 : 1.0; q.m1_efloor = desc->m1_efloor;
  q.m1_tol = desc->m1_tol > 0.0 ? desc->m1_tol : 1e-13; q.m1_mb = desc->m1_mb; q.m1_maxit = desc->m1_maxit > 0 ? desc->m1_maxit : 30;
  for (int i = 0; i < 3; ++i) q.m1_species_scale[i] = desc->m1_species_scale[i];
  q.m1_odd_even = desc->m1_odd_even; q.m1_arad = desc->m1_arad; q.m1_oe_guard = desc->m1_oe_guard;
  q.recon_kind = desc->recon_kind; q.weno_eps = desc->weno_eps; q.les_C_M = desc->les_C_M; q.les_C_N = desc->les_C_N; q.les_C_Y = desc->les_C_Y; q.les_C_T = desc->les_C_T;
  p->d_counts = nullptr;
  if (cudaMalloc(&p->d_counts, 48 * sizeof(unsigned long long)) != cudaSuccess) { delete p; return MHD_E_CUDA; }
  if (cudaMemset(p->d_counts, 0, 48 * sizeof(unsigned long long)) != cudaSuccess) { cudaFree(p->d_counts); delete p; return MHD_E_CUDA; }
  *out = p;
  return MHD_OK;
}

void mhd_patch_destroy(mhd_patch* p) {
  if (!p) return;
  for (auto& e : p->events) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  for (auto& e : p->pool) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  if (p->d_counts) cudaFree(p->d_counts);
  delete p;
}

int mhd_patch_bind(mhd_patch* p, int slot, void* dev_ptr, size_t field_stride) {
  if (!p || slot < 0 || slot >= MHD_NSLOTS || !dev_ptr) return MHD_E_ARG;
  if (field_stride < (size_t)p->dims.npts) return MHD_E_ARG;
  p->slot[slot].ptr = dev_ptr;
  p->slot[slot].stride = field_stride;
  return MHD_OK;
}

int mhd_fill_ghosts(mhd_patch* p, int slot_state, const int bc[6], void* stream) {
  if (!p || !bc) return MHD_E_ARG;
  const int n[3] = {p->dims.nx, p->dims.ny, p->dims.nz};
  bool halo = false;
  for (int a = 0; a < 6; ++a) {
    if (bc[a] < 0 || bc[a] > 2) return MHD_E_ARG;
    if (bc[a] != 1 && n[a / 2] < p->dims.ng) return MHD_E_ARG;      // a wrap by n must land on an interior point
    halo = halo || bc[a] == 2;
  }
  if (slot_state < 0 || slot_state >= MHD_NSLOTS || slot_state == MHD_SLOT_FLAGS) return MHD_E_ARG;
  if (!slot_ok(p, slot_state)) return MHD_E_UNBOUND;
  cudaStream_t s = (cudaStream_t)stream;
  const Slot& sl = p->slot[slot_state];
  unsigned long long *mine[27], *theirs[27];
  int nw = 0;
  if (halo) {
    // every direction whose non-zero components all cross a neighbour face needs the neighbour's array (faces, and the edges and
    // corners shared by two or three neighbour faces)
    for (int q = 0; q < 27; ++q) {
      const int dd[3] = {q % 3 - 1, (q / 3) % 3 - 1, q / 9 - 1};
      bool need = q != 13;
      for (int a = 0; a < 3; ++a) if (dd[a] != 0 && bc[2 * a + (dd[a] > 0)] != 2) need = false;
      if (!need) continue;
      if (!sl.peer[q]) return MHD_E_UNBOUND;
      if (p->peer_word[q]) { theirs[nw] = p->peer_word[q]; mine[nw] = p->d_counts + 16 + q; ++nw; }
    }
  }
  Timed tm(p, 0, s);
  // two-phase ordering against the neighbours (only when epoch words were registered: patches driven from one stream need none):
  // "my interior is final" -> all neighbours say so -> fill (reads their interiors) -> "I have read" -> all neighbours have read
  if (nw) {
    const unsigned long long e = ++p->halo_epoch;
    if (launch_halo_signal(theirs, nw, e, s) != cudaSuccess || launch_halo_wait(mine, nw, e, p->d_counts + 43, s) != cudaSuccess) return MHD_E_CUDA;
  }
  if (launch_fill_ghosts(p->dims, dptr(p, slot_state), sl.stride, slot_fields(slot_state), bc, halo ? &sl : nullptr, s) != cudaSuccess) return MHD_E_CUDA;
  if (nw) {
    const unsigned long long e = ++p->halo_epoch;
    if (launch_halo_signal(theirs, nw, e, s) != cudaSuccess || launch_halo_wait(mine, nw, e, p->d_counts + 43, s) != cudaSuccess) return MHD_E_CUDA;
  }
  return MHD_OK;
}

static int dir_index(const int dir[3]) {
  if (!dir) return -1;
  for (int a = 0; a < 3; ++a) if (dir[a] < -1 || dir[a] > 1) return -1;
  const int q = (dir[0] + 1) + 3 * (dir[1] + 1) + 9 * (dir[2] + 1);
  return q == 13 ? -1 : q;
}

int mhd_patch_set_neighbor(mhd_patch* p, int slot, const int dir[3], const void* peer_dev_ptr, size_t peer_field_stride) {
  const int q = dir_index(dir);
  if (!p || q < 0 || slot < 0 || slot >= MHD_NSLOTS || slot == MHD_SLOT_FLAGS) return MHD_E_ARG;
  if (peer_dev_ptr && peer_field_stride < (size_t)p->dims.npts) return MHD_E_ARG;
  p->slot[slot].peer[q] = (const double*)peer_dev_ptr;          // NULL clears the entry
  p->slot[slot].peer_stride[q] = peer_field_stride;
  return MHD_OK;
}

void* mhd_patch_halo_words(mhd_patch* p) { return p ? (void*)(p->d_counts + 16) : nullptr; }

int mhd_patch_set_neighbor_word(mhd_patch* p, const int dir[3], void* peer_words) {
  const int q = dir_index(dir);
  if (!p || q < 0) return MHD_E_ARG;
  // the neighbour in direction q sees this patch in direction 26 - q: that is the word of its array this patch signals
  p->peer_word[q] = peer_words ? (unsigned long long*)peer_words + (26 - q) : nullptr;
  return MHD_OK;
}

// ---- CUDA IPC helpers for one process per GPU: a device pointer inside any allocation (e.g. a torch tensor of the caching allocator)
// is exported as the allocation's handle plus the pointer's offset in it
int mhd_ipc_export(const void* dev_ptr, unsigned char handle[64], size_t* offset) {
  if (!dev_ptr || !handle || !offset) return MHD_E_ARG;
  typedef int (*RangeFn)(unsigned long long*, size_t*, unsigned long long);
  static RangeFn range = nullptr;
  if (!range) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess) return MHD_E_CUDA;
    range = (RangeFn)fn;
  }
  unsigned long long base = 0;
  size_t size = 0;
  if (range(&base, &size, (unsigned long long)(uintptr_t)dev_ptr) != 0) return MHD_E_CUDA;
  static_assert(sizeof(cudaIpcMemHandle_t) == 64, "handle size");
  cudaIpcMemHandle_t h;
  if (cudaIpcGetMemHandle(&h, (void*)(uintptr_t)base) != cudaSuccess) { cudaGetLastError(); return MHD_E_CUDA; }
  memcpy(handle, &h, 64);
  *offset = (size_t)((unsigned long long)(uintptr_t)dev_ptr - base);
  return MHD_OK;
}

int mhd_ipc_import(const unsigned char handle[64], size_t offset, void** dev_ptr) {
  if (!handle || !dev_ptr) return MHD_E_ARG;
  cudaIpcMemHandle_t h;
  memcpy(&h, handle, 64);
  void* base = nullptr;
  if (cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) { cudaGetLastError(); return MHD_E_CUDA; }
  *dev_ptr = (char*)base + offset;
  return MHD_OK;
}

int mhd_ipc_close(void* dev_ptr, size_t offset) {
  if (!dev_ptr) return MHD_E_ARG;
  return cudaIpcCloseMemHandle((char*)dev_ptr - offset) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_con2prim(mhd_patch* p, int slot_state, int slot_prim, int slot_flags, void* stream) {
  if (!p || !is_state_slot(slot_state) || slot_prim != MHD_SLOT_P || slot_flags != MHD_SLOT_FLAGS) return MHD_E_ARG;
  if (!slot_ok(p, slot_state) || !slot_ok(p, slot_prim) || !slot_ok(p, slot_flags)) return MHD_E_UNBOUND;
  Timed tm(p, 1, (cudaStream_t)stream);
  return launch_con2prim(p->dims, p->par, dptr(p, slot_state), p->slot[slot_state].stride, dptr(p, slot_prim), p->slot[slot_prim].stride,
                         (uint8_t*)p->slot[slot_flags].ptr, (double*)(p->d_counts + 8), (cudaStream_t)stream) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_prim2con(mhd_patch* p, int slot_state, int slot_prim, void* stream) {
  if (!p || !is_state_slot(slot_state) || slot_prim != MHD_SLOT_P) return MHD_E_ARG;
  if (!slot_ok(p, slot_state) || !slot_ok(p, slot_prim)) return MHD_E_UNBOUND;
  return launch_prim2con(p->dims, p->par, dptr(p, slot_state), p->slot[slot_state].stride, dptr(p, slot_prim), p->slot[slot_prim].stride,
                         (cudaStream_t)stream) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_rhs(mhd_patch* p, int slot_state, int slot_prim, int slot_rhs, void* stream) {
  if (!p || !is_state_slot(slot_state) || slot_prim != MHD_SLOT_P || !is_state_slot(slot_rhs) || slot_rhs == slot_state) return MHD_E_ARG;
  if (!slot_ok(p, slot_state) || !slot_ok(p, slot_prim) || !slot_ok(p, slot_rhs) || !slot_ok(p, MHD_SLOT_WORK)) return MHD_E_UNBOUND;
  return rhs_impl(p, slot_state, slot_prim, slot_rhs, Fuse(), (cudaStream_t)stream);
}

int mhd_les_flux(mhd_patch* p, int slot_state, int slot_prim, void* stream) {
  if (!p || !is_state_slot(slot_state) || slot_prim != MHD_SLOT_P) return MHD_E_ARG;
  if (!les_on(p->par)) return MHD_E_ARG;
  if (!slot_ok(p, slot_state) || !slot_ok(p, slot_prim)) return MHD_E_UNBOUND;
  return les_impl(p, slot_state, slot_prim, (cudaStream_t)stream);
}

int mhd_rk_stage(mhd_patch* p, const mhd_tableau* t, int stage, double dt, void* stream) {
  if (!p || !t || !t->a_expl || !t->w_expl || t->stages < 1 || t->stages > MHD_MAX_STAGES || stage < 0 || stage > t->stages) return MHD_E_ARG;
  if (!slot_ok(p, MHD_SLOT_U) || !slot_ok(p, MHD_SLOT_U0)) return MHD_E_UNBOUND;
  cudaStream_t s = (cudaStream_t)stream;
  Timed tm(p, 6, s);
  if (stage == 0)
    return launch_copy_fields(p->dims, MHD_NSTATE, dptr(p, MHD_SLOT_U0), p->slot[MHD_SLOT_U0].stride, dptr(p, MHD_SLOT_U), p->slot[MHD_SLOT_U].stride, s) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
  const double* coef = stage < t->stages ? t->a_expl + (size_t)stage * t->stages : t->w_expl;
  const int nmax = stage < t->stages ? stage : t->stages;
  const double* Kp[MHD_MAX_STAGES];
  size_t sk[MHD_MAX_STAGES];
  double c[MHD_MAX_STAGES];
  int nk = 0;
  for (int j = 0; j < nmax; ++j) {
    if (coef[j] == 0.0) continue;
    if (!slot_ok(p, MHD_SLOT_K1 + j)) return MHD_E_UNBOUND;
    Kp[nk] = dptr(p, MHD_SLOT_K1 + j); sk[nk] = p->slot[MHD_SLOT_K1 + j].stride; c[nk] = coef[j]; ++nk;
  }
  if (nk == 0)   // U <- U0
    return launch_copy_fields(p->dims, MHD_NSTATE, dptr(p, MHD_SLOT_U), p->slot[MHD_SLOT_U].stride, dptr(p, MHD_SLOT_U0), p->slot[MHD_SLOT_U0].stride, s) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
  return launch_rk_combine(p->dims, MHD_NSTATE, dptr(p, MHD_SLOT_U), p->slot[MHD_SLOT_U].stride, dptr(p, MHD_SLOT_U0), p->slot[MHD_SLOT_U0].stride,
                           nk, Kp, sk, c, dt, s) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_advance(mhd_patch* p, const mhd_tableau* t, const int bc[6], double dt, int n_steps, void* stream) {
  if (!p || !t || !bc || n_steps < 0) return MHD_E_ARG;
  return stage_sequence(p, t, bc, dt, n_steps, (cudaStream_t)stream);
}

// packed host array <-> slot (field stride of the slot may exceed the packed one)
static bool copy_fields(double* dst, size_t sd, const double* src, size_t ss, int nfields, size_t n, cudaMemcpyKind kind, cudaStream_t s) {
  if (sd == n && ss == n) return cudaMemcpyAsync(dst, src, n * nfields * sizeof(double), kind, s) == cudaSuccess;
  for (int f = 0; f < nfields; ++f)
    if (cudaMemcpyAsync(dst + f * sd, src + f * ss, n * sizeof(double), kind, s) != cudaSuccess) return false;
  return true;
}

int mhd_advance_imex_host(mhd_patch* p, const mhd_tableau* t, const int bc[6], double dt, int n_steps, double* host_U, double* host_V,
                          uint8_t* host_flags, void* stream) {
  if (!p || !t || !bc || !host_U || !host_V || n_steps < 0) return MHD_E_ARG;
  if (p->desc.n_species != 3) return MHD_E_UNSUPPORTED;
  if (!slot_ok(p, MHD_SLOT_U) || !slot_ok(p, MHD_SLOT_V) || !slot_ok(p, MHD_SLOT_FLAGS)) return MHD_E_UNBOUND;
  cudaStream_t s = (cudaStream_t)stream;
  const size_t n = (size_t)p->dims.npts;
  if (!copy_fields(dptr(p, MHD_SLOT_U), p->slot[MHD_SLOT_U].stride, host_U, n, MHD_NSTATE, n, cudaMemcpyHostToDevice, s)) return MHD_E_CUDA;
  if (!copy_fields(dptr(p, MHD_SLOT_V), p->slot[MHD_SLOT_V].stride, host_V, n, MHD_NM1, n, cudaMemcpyHostToDevice, s)) return MHD_E_CUDA;
  const int rc = mhd_advance_imex(p, t, bc, dt, n_steps, stream);
  if (rc != MHD_OK) return rc;
  if (!copy_fields(host_U, n, dptr(p, MHD_SLOT_U), p->slot[MHD_SLOT_U].stride, MHD_NSTATE, n, cudaMemcpyDeviceToHost, s)) return MHD_E_CUDA;
  if (!copy_fields(host_V, n, dptr(p, MHD_SLOT_V), p->slot[MHD_SLOT_V].stride, MHD_NM1, n, cudaMemcpyDeviceToHost, s)) return MHD_E_CUDA;
  if (host_flags && cudaMemcpyAsync(host_flags, p->slot[MHD_SLOT_FLAGS].ptr, n, cudaMemcpyDeviceToHost, s) != cudaSuccess) return MHD_E_CUDA;
  return cudaStreamSynchronize(s) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_advance_host(mhd_patch* p, const mhd_tableau* t, const int bc[6], double dt, int n_steps, double* host_U, uint8_t* host_flags, void* stream) {
  if (!p || !t || !bc || !host_U || n_steps < 0) return MHD_E_ARG;
  if (!slot_ok(p, MHD_SLOT_U) || !slot_ok(p, MHD_SLOT_FLAGS)) return MHD_E_UNBOUND;
  cudaStream_t s = (cudaStream_t)stream;
  const size_t n = (size_t)p->dims.npts, su = p->slot[MHD_SLOT_U].stride;
  double* U = dptr(p, MHD_SLOT_U);
  if (su == n) {
    if (cudaMemcpyAsync(U, host_U, n * MHD_NSTATE * sizeof(double), cudaMemcpyHostToDevice, s) != cudaSuccess) return MHD_E_CUDA;
  } else {
    for (int f = 0; f < MHD_NSTATE; ++f)
      if (cudaMemcpyAsync(U + f * su, host_U + f * n, n * sizeof(double), cudaMemcpyHostToDevice, s) != cudaSuccess) return MHD_E_CUDA;
  }
  const int rc = stage_sequence(p, t, bc, dt, n_steps, s);
  if (rc != MHD_OK) return rc;
  if (su == n) {
    if (cudaMemcpyAsync(host_U, U, n * MHD_NSTATE * sizeof(double), cudaMemcpyDeviceToHost, s) != cudaSuccess) return MHD_E_CUDA;
  } else {
    for (int f = 0; f < MHD_NSTATE; ++f)
      if (cudaMemcpyAsync(host_U + f * n, U + f * su, n * sizeof(double), cudaMemcpyDeviceToHost, s) != cudaSuccess) return MHD_E_CUDA;
  }
  if (host_flags && cudaMemcpyAsync(host_flags, p->slot[MHD_SLOT_FLAGS].ptr, n, cudaMemcpyDeviceToHost, s) != cudaSuccess) return MHD_E_CUDA;
  return cudaStreamSynchronize(s) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_m1_implicit(mhd_patch* p, int slot_V, int slot_R, double adt, void* stream) {
  if (!p || !is_m1_slot(slot_V) || !is_m1_slot(slot_R) || slot_V == slot_R || !(adt >= 0.0)) return MHD_E_ARG;
  if (p->desc.n_species != 3) return MHD_E_UNSUPPORTED;
  if (!slot_ok(p, slot_V) || !slot_ok(p, slot_R) || !slot_ok(p, MHD_SLOT_U) || !slot_ok(p, MHD_SLOT_P) || !slot_ok(p, MHD_SLOT_FLAGS)) return MHD_E_UNBOUND;
  Timed tm(p, 11, (cudaStream_t)stream);
  return launch_m1_implicit(p->dims, p->par, dptr(p, MHD_SLOT_U), p->slot[MHD_SLOT_U].stride, dptr(p, MHD_SLOT_P), p->slot[MHD_SLOT_P].stride,
                            dptr(p, slot_V), p->slot[slot_V].stride, dptr(p, slot_R), p->slot[slot_R].stride, adt,
                            (uint8_t*)p->slot[MHD_SLOT_FLAGS].ptr, (cudaStream_t)stream) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_m1_rhs(mhd_patch* p, int slot_V, int slot_KV, void* stream) {
  if (!p || !is_m1_slot(slot_V) || !is_m1_slot(slot_KV) || slot_V == slot_KV) return MHD_E_ARG;
  if (p->desc.n_species != 3) return MHD_E_UNSUPPORTED;
  if (!slot_ok(p, slot_V) || !slot_ok(p, slot_KV) || !slot_ok(p, MHD_SLOT_U) || !slot_ok(p, MHD_SLOT_P) || !slot_ok(p, MHD_SLOT_M1WORK)) return MHD_E_UNBOUND;
  cudaStream_t s = (cudaStream_t)stream;
  const double* U = dptr(p, MHD_SLOT_U);
  const size_t su = p->slot[MHD_SLOT_U].stride, sw = p->slot[MHD_SLOT_M1WORK].stride;
  { Timed tm(p, 9, s);
    if (launch_m1_point(p->dims, p->par, U, su, dptr(p, MHD_SLOT_P), p->slot[MHD_SLOT_P].stride, dptr(p, slot_V), p->slot[slot_V].stride,
                        dptr(p, MHD_SLOT_M1WORK), sw, s) != cudaSuccess) return MHD_E_CUDA; }
  Timed tm(p, 10, s);
  return launch_m1_div(p->dims, p->par, U, su, dptr(p, slot_V), p->slot[slot_V].stride, dptr(p, MHD_SLOT_M1WORK), sw, dptr(p, slot_KV), p->slot[slot_KV].stride, s)
         == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_m1_backreaction(mhd_patch* p, int slot_R, int slot_K, void* stream) {
  if (!p || !is_m1_slot(slot_R) || !is_state_slot(slot_K)) return MHD_E_ARG;
  if (p->desc.n_species != 3) return MHD_E_UNSUPPORTED;
  if (!slot_ok(p, slot_R) || !slot_ok(p, slot_K)) return MHD_E_UNBOUND;
  Timed tm(p, 11, (cudaStream_t)stream);
  return launch_m1_backreact(p->dims, p->par, dptr(p, slot_R), p->slot[slot_R].stride, dptr(p, slot_K), p->slot[slot_K].stride, (cudaStream_t)stream)
         == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_m1_gravity(mhd_patch* p, int slot_V, int slot_K, void* stream) {
  if (!p || !is_m1_slot(slot_V) || !is_state_slot(slot_K)) return MHD_E_ARG;
  if (p->desc.n_species != 3) return MHD_E_UNSUPPORTED;
  if (!slot_ok(p, slot_V) || !slot_ok(p, slot_K) || !slot_ok(p, MHD_SLOT_U) || !slot_ok(p, MHD_SLOT_M1WORK)) return MHD_E_UNBOUND;
  Timed tm(p, 11, (cudaStream_t)stream);
  return launch_m1_gravity(p->dims, p->par, dptr(p, MHD_SLOT_U), p->slot[MHD_SLOT_U].stride, dptr(p, slot_V), p->slot[slot_V].stride,
                           dptr(p, MHD_SLOT_M1WORK), p->slot[MHD_SLOT_M1WORK].stride, dptr(p, slot_K), p->slot[slot_K].stride, (cudaStream_t)stream)
         == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

// V <- V0 + dt (sum_j ce[j] KV_j + sum_j ci[j] R_j), j < nj
static int m1_combine(mhd_patch* p, int nj, const double* ce, const double* ci, double dt, cudaStream_t s) {
  const double* Kp[MHD_MAX_STAGES];
  size_t sk[MHD_MAX_STAGES];
  double c[MHD_MAX_STAGES];
  int nk = 0;
  for (int pass = 0; pass < 2; ++pass)
    for (int j = 0; j < nj; ++j) {
      const double cj = pass == 0 ? ce[j] : ci[j];
      if (cj == 0.0) continue;
      const int slot = (pass == 0 ? MHD_SLOT_KV1 : MHD_SLOT_R1) + j;
      if (!slot_ok(p, slot)) return MHD_E_UNBOUND;
      if (nk == MHD_MAX_STAGES) return MHD_E_ARG;
      Kp[nk] = dptr(p, slot); sk[nk] = p->slot[slot].stride; c[nk] = cj; ++nk;
    }
  Timed tm(p, 6, s);
  if (nk == 0)
    return launch_copy_fields(p->dims, MHD_NM1, dptr(p, MHD_SLOT_V), p->slot[MHD_SLOT_V].stride, dptr(p, MHD_SLOT_V0), p->slot[MHD_SLOT_V0].stride, s) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
  return launch_rk_combine(p->dims, MHD_NM1, dptr(p, MHD_SLOT_V), p->slot[MHD_SLOT_V].stride, dptr(p, MHD_SLOT_V0), p->slot[MHD_SLOT_V0].stride,
                           nk, Kp, sk, c, dt, s) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_advance_imex(mhd_patch* p, const mhd_tableau* t, const int bc[6], double dt, int n_steps, void* stream) {
  if (!p || !t || !bc || n_steps < 0 || !t->a_expl || !t->w_expl || !t->a_impl || !t->w_impl || t->stages < 1 || t->stages > MHD_MAX_STAGES) return MHD_E_ARG;
  if (p->desc.n_species != 3) return MHD_E_UNSUPPORTED;
  for (int sl : {MHD_SLOT_U, MHD_SLOT_U0, MHD_SLOT_P, MHD_SLOT_FLAGS, MHD_SLOT_V, MHD_SLOT_V0}) if (!slot_ok(p, sl)) return MHD_E_UNBOUND;
  cudaStream_t s = (cudaStream_t)stream;
  const int q = t->stages;
  int rc;
#define CK(call) if ((rc = (call)) != MHD_OK) return rc
  for (int step = 0; step < n_steps; ++step) {
    CK(mhd_fill_ghosts(p, MHD_SLOT_U, bc, s));
    CK(mhd_con2prim(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_FLAGS, s));
    CK(mhd_fill_ghosts(p, MHD_SLOT_V, bc, s));
    CK(mhd_rk_stage(p, t, 0, dt, s));                                                    // U0 <- U
    { Timed tm(p, 6, s);
      if (launch_copy_fields(p->dims, MHD_NM1, dptr(p, MHD_SLOT_V0), p->slot[MHD_SLOT_V0].stride, dptr(p, MHD_SLOT_V), p->slot[MHD_SLOT_V].stride, s) != cudaSuccess) return MHD_E_CUDA; }
    for (int st = 0; st < q; ++st) {
      if (st > 0) {                                                                      // explicit intermediate values (C3)
        CK(mhd_rk_stage(p, t, st, dt, s));
        CK(m1_combine(p, st, t->a_expl + (size_t)st * q, t->a_impl + (size_t)st * q, dt, s));
        CK(mhd_fill_ghosts(p, MHD_SLOT_U, bc, s));
        CK(mhd_con2prim(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_FLAGS, s));
        CK(mhd_fill_ghosts(p, MHD_SLOT_V, bc, s));
      }
      CK(mhd_m1_implicit(p, MHD_SLOT_V, MHD_SLOT_R1 + st, t->a_impl[(size_t)st * q + st] * dt, s));   // (C4)
      CK(mhd_m1_rhs(p, MHD_SLOT_V, MHD_SLOT_KV1 + st, s));                            // also leaves P_ij of V^(i) in the M1 work slot
      CK(mhd_rhs(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_K1 + st, s));
      CK(mhd_m1_backreaction(p, MHD_SLOT_R1 + st, MHD_SLOT_K1 + st, s));
      CK(mhd_m1_gravity(p, MHD_SLOT_V, MHD_SLOT_K1 + st, s));
    }
    CK(mhd_rk_stage(p, t, q, dt, s));
    CK(m1_combine(p, q, t->w_expl, t->w_impl, dt, s));
  }
  CK(mhd_fill_ghosts(p, MHD_SLOT_U, bc, s));
  CK(mhd_con2prim(p, MHD_SLOT_U, MHD_SLOT_P, MHD_SLOT_FLAGS, s));
  return mhd_fill_ghosts(p, MHD_SLOT_V, bc, s);
#undef CK
}

// ---- AMR transfer operators on a patch pair
int mhd_prolong(mhd_patch* coarse, int slot_c, mhd_patch* fine, int slot_f, const int origin[3], const int lo[3], const int hi[3], void* stream) {
  if (!coarse || !fine || !origin || !lo || !hi || coarse == fine) return MHD_E_ARG;
  if (slot_c < 0 || slot_c >= MHD_NSLOTS || slot_f < 0 || slot_f >= MHD_NSLOTS || slot_c == MHD_SLOT_FLAGS || slot_f == MHD_SLOT_FLAGS) return MHD_E_ARG;
  if (slot_fields(slot_c) != slot_fields(slot_f)) return MHD_E_ARG;
  if (!slot_ok(coarse, slot_c) || !slot_ok(fine, slot_f)) return MHD_E_UNBOUND;
  const Dims &dc = coarse->dims, &df = fine->dims;
  const int mf[3] = {df.mx, df.my, df.mz}, mc[3] = {dc.mx, dc.my, dc.mz};
  for (int a = 0; a < 3; ++a) {
    if (lo[a] < 0 || hi[a] > mf[a] || hi[a] < lo[a]) return MHD_E_ARG;
    if (hi[a] == lo[a]) return MHD_OK;
    // every coarse point the box needs (offsets -2..3 around a midpoint, the point itself under a coincident point) must exist
    for (int e = 0; e < 2; ++e) {
      const int af = (e == 0 ? lo[a] : hi[a] - 1) - df.ng;
      const int hfl = af >= 0 ? af / 2 : -((-af + 1) / 2);
      const int c = origin[a] + hfl + dc.ng, odd = af - 2 * hfl;
      // a box of more than one point holds both parities: test the wider stencil unless the box is a single point
      const bool wide = odd || hi[a] - lo[a] > 1;
      if (c - (wide ? 2 : 0) < 0 || c + (wide ? 3 : 0) >= mc[a]) return MHD_E_ARG;
    }
  }
  return launch_prolong(dc, dptr(coarse, slot_c), coarse->slot[slot_c].stride, df, dptr(fine, slot_f), fine->slot[slot_f].stride, slot_fields(slot_c),
                        origin, lo, hi, (cudaStream_t)stream) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_restrict(mhd_patch* fine, int slot_f, mhd_patch* coarse, int slot_c, const int origin[3], void* stream) {
  if (!coarse || !fine || !origin || coarse == fine) return MHD_E_ARG;
  if (slot_c < 0 || slot_c >= MHD_NSLOTS || slot_f < 0 || slot_f >= MHD_NSLOTS || slot_c == MHD_SLOT_FLAGS || slot_f == MHD_SLOT_FLAGS) return MHD_E_ARG;
  if (slot_fields(slot_c) != slot_fields(slot_f)) return MHD_E_ARG;
  if (!slot_ok(coarse, slot_c) || !slot_ok(fine, slot_f)) return MHD_E_UNBOUND;
  const Dims &dc = coarse->dims, &df = fine->dims;
  const int nf[3] = {df.nx, df.ny, df.nz}, mc[3] = {dc.mx, dc.my, dc.mz};
  for (int a = 0; a < 3; ++a)
    if (origin[a] + dc.ng < 0 || origin[a] + (nf[a] - 1) / 2 + dc.ng >= mc[a]) return MHD_E_ARG;
  return launch_restrict(df, dptr(fine, slot_f), fine->slot[slot_f].stride, dc, dptr(coarse, slot_c), coarse->slot[slot_c].stride, slot_fields(slot_c),
                         origin, (cudaStream_t)stream) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_dense_weights(int scheme, double theta, int deriv, double b[4]) {
  if (!b || (scheme != 0 && scheme != 1) || deriv < 0 || deriv > 3) return MHD_E_ARG;
  // coefficients of theta^1, theta^2, theta^3 of b_j(theta): Eq. (58) RK(4,4), Eq. (59) SSP-RK(3,3)
  static const double rk4[4][3] = {{1.0, -1.5, 2.0 / 3.0}, {0.0, 1.0, -2.0 / 3.0}, {0.0, 1.0, -2.0 / 3.0}, {0.0, -0.5, 2.0 / 3.0}};
  static const double ssp3[4][3] = {{1.0, -5.0 / 6.0, 0.0}, {0.0, 1.0 / 6.0, 0.0}, {0.0, 4.0 / 6.0, 0.0}, {0.0, 0.0, 0.0}};
  const double (*p)[3] = scheme == 0 ? rk4 : ssp3;
  const double t = theta;
  for (int j = 0; j < 4; ++j) {
    const double c1 = p[j][0], c2 = p[j][1], c3 = p[j][2];
    b[j] = deriv == 0 ? t * (c1 + t * (c2 + t * c3)) : deriv == 1 ? c1 + t * (2.0 * c2 + 3.0 * t * c3) : deriv == 2 ? 2.0 * c2 + 6.0 * t * c3 : 6.0 * c3;
  }
  return scheme == 0 ? 4 : 3;
}

int mhd_dense_output(mhd_patch* p, int scheme, double theta, double dt, int deriv, int slot_out, void* stream) {
  double b[4];
  const int s = mhd_dense_weights(scheme, theta, deriv, b);
  if (!p || s < 0 || !(dt > 0.0) || !is_state_slot(slot_out) || slot_out == MHD_SLOT_U0) return MHD_E_ARG;
  if (!slot_ok(p, slot_out) || !slot_ok(p, MHD_SLOT_U0)) return MHD_E_UNBOUND;
  const double* K[4]; size_t sk[4]; double c[4];
  for (int j = 0; j < s; ++j) {
    if (slot_out == MHD_SLOT_K1 + j) return MHD_E_ARG;
    if (!slot_ok(p, MHD_SLOT_K1 + j)) return MHD_E_UNBOUND;
    K[j] = dptr(p, MHD_SLOT_K1 + j); sk[j] = p->slot[MHD_SLOT_K1 + j].stride;
    c[j] = b[j] * dt / pow(dt, deriv);                     // k_j = dt K_j; Eq. (57): dt^-m
  }
  Timed tm(p, 6, (cudaStream_t)stream);
  return launch_dense(p->dims, MHD_NSTATE, dptr(p, slot_out), p->slot[slot_out].stride, dptr(p, MHD_SLOT_U0), p->slot[MHD_SLOT_U0].stride, s, K, sk, c,
                      deriv == 0, (cudaStream_t)stream) == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}

int mhd_patch_status(mhd_patch* p, int slot_flags, mhd_status* out, void* stream) {
  if (!p || !out || slot_flags != MHD_SLOT_FLAGS) return MHD_E_ARG;
  if (!slot_ok(p, slot_flags)) return MHD_E_UNBOUND;
  cudaStream_t s = (cudaStream_t)stream;
  if (launch_count_flags(p->dims, (const uint8_t*)p->slot[slot_flags].ptr, p->d_counts, s) != cudaSuccess) return MHD_E_CUDA;
  unsigned long long h[8], hto = 0;
  if (cudaMemcpyAsync(h, p->d_counts, sizeof(h), cudaMemcpyDeviceToHost, s) != cudaSuccess) return MHD_E_CUDA;
  if (cudaMemcpyAsync(&hto, p->d_counts + 43, sizeof(hto), cudaMemcpyDeviceToHost, s) != cudaSuccess) return MHD_E_CUDA;
  if (cudaStreamSynchronize(s) != cudaSuccess) return MHD_E_CUDA;
  out->n_points = (unsigned long long)p->dims.npts;
  out->n_atmo = h[0]; out->n_eps_lo = h[1]; out->n_eps_hi = h[2]; out->n_vmax = h[3];
  out->n_ye = h[4]; out->n_fatal = h[5]; out->n_noconv = h[6]; out->n_m1fix = h[7];
  out->halo_timeout = hto;
  return MHD_OK;
}

int mhd_patch_profile(mhd_patch* p, int enable) {
  if (!p) return MHD_E_ARG;
  p->profiling = enable != 0;
  // events are created here, outside any timed region: enough pairs for a few RK steps of the longest stage sequence
  while (enable && p->pool.size() < 256) {
    mhd_patch::Ev ev;
    if (cudaEventCreate(&ev.a) != cudaSuccess || cudaEventCreate(&ev.b) != cudaSuccess) return MHD_E_CUDA;
    ev.cls = 0;
    p->pool.push_back(ev);
  }
  return MHD_OK;
}

int mhd_patch_profile_read(mhd_patch* p, double ms[MHD_NKERNELS], unsigned long long launches[MHD_NKERNELS], void* stream) {
  if (!p || !ms || !launches) return MHD_E_ARG;
  if (cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) return MHD_E_CUDA;
  for (int c = 0; c < MHD_NKERNELS; ++c) { ms[c] = 0.0; launches[c] = 0; }
  for (auto& e : p->events) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, e.a, e.b) != cudaSuccess) return MHD_E_CUDA;
    ms[e.cls] += t; launches[e.cls] += 1;
    p->pool.push_back(e);
  }
  p->events.clear();
  return MHD_OK;
}

double mhd_probe_fp64_flops(void* stream) { return probe_fp64((cudaStream_t)stream); }

const char* mhd_strerror(int code) {
  switch (code) {
    case MHD_OK: return "ok";
    case MHD_E_ARG: return "invalid argument";
    case MHD_E_UNBOUND: return "slot not bound";
    case MHD_E_CUDA: return "CUDA runtime error";
    case MHD_E_UNSUPPORTED: return "feature not supported by this build";
    case MHD_E_TOO_LARGE: return "size beyond the fixed capacity of this allocation-free entry point";
    default: return "unknown error";
  }
}

}  // extern "C"
