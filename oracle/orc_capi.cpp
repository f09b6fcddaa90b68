// ORACLE (test infrastructure) — plain C entry points for the ctypes binding in oracle/__init__.py.
#include <cstring>
#include <string>
#include "orc.hpp"

using namespace orc;

namespace {
struct Handle { Params par; Grid grid; };

bool set_scalar(Params& p, const std::string& k, double v) {
#define D(name) if (k == #name) { p.name = v; return true; }
#define I(name) if (k == #name) { p.name = (int)v; return true; }
  I(eos_kind) D(eos_gamma) D(eos_gamma_th) I(n_pieces)
  D(kappa_z) D(kappa_c) D(kappa_2) D(eta_shift) D(f_alpha) D(f_beta) D(grav_G)
  D(sigma_ko_spacetime) D(sigma_ko_matter) D(c_b) D(kappa_b) D(mp5_alpha)
  D(rho_atmo) D(rho_cut) D(rho_low) D(alpha_bh) D(w_max) D(rho_max) D(eps_min) D(eps_max)
  D(ye_min) D(ye_max) D(ye_atmo) D(eps_atmo) D(T_atmo) I(c2p_maxit)
  D(m1_kappa0) D(m1_rho0) D(m1_efloor) D(m1_tol) D(m1_mb) I(m1_maxit) I(m1_odd_even) D(m1_arad) D(m1_oe_guard)
  I(recon_kind) D(weno_eps) D(les_C_M) D(les_C_N) D(les_C_Y) D(les_C_T)
  I(n_rho) I(n_T) I(n_ye) D(lr0) D(dlr) D(lT0) D(dlT) D(ye0) D(dye) D(tab_eps_shift) D(tab_h0)
#undef D
#undef I
  return false;
}
}  // namespace

#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

// thread count of the -fopenmp build (the outermost grid loops carry `#pragma omp parallel for`; the arithmetic of every point
// is unchanged). Returns the count in effect: always 1 in the plain build.
int orc_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
  return omp_get_max_threads();
#else
  (void)n;
  return 1;
#endif
}

void* orc_new() {
  Handle* h = new Handle();
  std::memset(&h->par, 0, sizeof(Params));
  std::memset(&h->grid, 0, sizeof(Grid));
  return h;
}
void orc_free(void* h) { delete (Handle*)h; }

int orc_set(void* h, const char* key, double v) { return set_scalar(((Handle*)h)->par, key, v) ? 0 : -1; }

int orc_set_array(void* hh, const char* key, const double* v, int n) {
  Params& p = ((Handle*)hh)->par;
  const std::string k = key;
  double* dst = nullptr;
  int cap = 8;
  if (k == "pp_K") dst = p.pp_K;
  else if (k == "pp_Gamma") dst = p.pp_Gamma;
  else if (k == "pp_rho") dst = p.pp_rho;
  else if (k == "beta0") { dst = p.beta0; cap = 3; }
  else if (k == "m1_species_scale") { dst = p.m1_species_scale; cap = 3; }
  if (!dst || n > cap) return -1;
  for (int i = 0; i < n; ++i) dst[i] = v[i];
  return 0;
}
// table pointers are borrowed (caller keeps the arrays alive)
void orc_set_table(void* hh, const double* logp, const double* loge, const double* cs2) {
  Params& p = ((Handle*)hh)->par;
  p.tab_logp = logp; p.tab_loge = loge; p.tab_cs2 = cs2;
}
void orc_finalize(void* hh) { eos_init(((Handle*)hh)->par); }

void orc_set_grid(void* hh, int nx, int ny, int nz, int ng, double dx, double dy, double dz) {
  ((Handle*)hh)->grid = Grid{nx, ny, nz, ng, dx, dy, dz};
}

void orc_fill_ghosts(void* hh, double* U, int nfields, const int* bc) { fill_ghosts(((Handle*)hh)->grid, U, nfields, bc); }
void orc_con2prim(void* hh, double* U, double* P, uint8_t* flags) { Handle* h = (Handle*)hh; con2prim(h->par, h->grid, U, P, flags); }
void orc_prim2con(void* hh, double* U, double* P) { Handle* h = (Handle*)hh; prim2con(h->par, h->grid, U, P); }
void orc_rhs(void* hh, const double* U, const double* P, double* K) { Handle* h = (Handle*)hh; rhs(h->par, h->grid, U, P, K); }
void orc_rhs_ccz4(void* hh, const double* U, const double* P, double* K) { Handle* h = (Handle*)hh; rhs_ccz4(h->par, h->grid, U, P, K); }
void orc_rhs_grmhd(void* hh, const double* U, const double* P, double* K) { Handle* h = (Handle*)hh; rhs_grmhd(h->par, h->grid, U, P, K); }
void orc_rhs_grmhd_flux(void* hh, const double* U, const double* P, double* K) { Handle* h = (Handle*)hh; rhs_grmhd_parts(h->par, h->grid, U, P, K, 1); }
void orc_rhs_grmhd_src(void* hh, const double* U, const double* P, double* K) { Handle* h = (Handle*)hh; rhs_grmhd_parts(h->par, h->grid, U, P, K, 2); }
void orc_rk_combine(void* hh, int nfields, double* Uout, const double* U0, int nk, const double* const* K, const double* coef, double dt) {
  rk_combine(((Handle*)hh)->grid, nfields, Uout, U0, nk, K, coef, dt);
}
void orc_evolve(void* hh, double* U, double* P, uint8_t* flags, const int* bc, int stages,
                const double* a_expl, const double* w_expl, double dt, int n_steps) {
  Handle* h = (Handle*)hh;
  evolve(h->par, h->grid, U, P, flags, bc, stages, a_expl, w_expl, dt, n_steps);
}

// ---- M1
void orc_m1_closure_point(double E, const double* F, const double* vu, double W, const double* gl, const double* gu, double* out16) {
  const M1Closure c = m1_closure_point(E, F, vu, W, (const double (*)[3])gl, (const double (*)[3])gu);
  out16[0] = c.xi; out16[1] = c.chi; out16[2] = c.J; out16[3] = c.Hn;
  for (int i = 0; i < 3; ++i) { out16[4 + i] = c.H[i]; for (int j = 0; j < 3; ++j) out16[7 + 3 * i + j] = c.P[i][j]; }
}
void orc_m1_JH(double E, const double* F, const double* vu, double W, const double* gl, const double* gu, double dthin, double dthick, double* out4) {
  m1_JH_appC(E, F, vu, W, (const double (*)[3])gl, (const double (*)[3])gu, dthin, dthick, out4[0], out4 + 1);
}
void orc_m1_jacobian(double E, const double* F, const double* vu, double W, const double* gl, const double* gu, double dthin, double dthick,
                     double alpha, double ka, double ks, double* out16) {
  m1_jacobian(E, F, vu, W, (const double (*)[3])gl, (const double (*)[3])gu, dthin, dthick, alpha, ka, ks, (double (*)[4])out16);
}
int orc_m1_implicit_point(void* hh, int species, const double* Vstar, double adt, double alpha, const double* vu, double W, double rho, double T,
                          const double* gl, const double* gu, double* V, double* R) {
  return m1_implicit_point(((Handle*)hh)->par, species, Vstar, adt, alpha, vu, W, rho, T, (const double (*)[3])gl, (const double (*)[3])gu, V, R);
}
void orc_m1_rhs(void* hh, const double* U, const double* P, const double* V, double* KV) { Handle* h = (Handle*)hh; m1_rhs(h->par, h->grid, U, P, V, KV); }
void orc_m1_implicit(void* hh, const double* U, const double* P, double* V, double* R, double adt, uint8_t* flags) {
  Handle* h = (Handle*)hh; m1_implicit(h->par, h->grid, U, P, V, R, adt, flags);
}
void orc_m1_backreaction(void* hh, const double* U, const double* P, const double* R, double* K) { Handle* h = (Handle*)hh; m1_backreaction(h->par, h->grid, U, P, R, K); }
void orc_m1_gravity(void* hh, const double* U, const double* P, const double* V, double* K) { Handle* h = (Handle*)hh; m1_gravity(h->par, h->grid, U, P, V, K); }
void orc_evolve_imex(void* hh, double* U, double* V, double* P, uint8_t* flags, const int* bc, int stages, const double* ae, const double* we,
                     const double* ai, const double* wi, double dt, int n_steps) {
  Handle* h = (Handle*)hh;
  evolve_imex(h->par, h->grid, U, V, P, flags, bc, stages, ae, we, ai, wi, dt, n_steps);
}

// ---- LES (App. A)
void orc_les_flux(void* hh, const double* U, const double* P, double* L9, double* A26) { Handle* h = (Handle*)hh; les_flux(h->par, h->grid, U, P, L9, A26); }
void orc_les_HM_point(const double* a26, const double* da3x26, const double* gu9, double p, double* HM9) {
  les_HM_point(a26, (const double (*)[LES_NAUX])da3x26, (const double (*)[3])gu9, p, (double (*)[3])HM9);
}
void orc_les_H_point(const double* a, const double* da, const double* gu9, const double* gl9, double sqrtg, double p, double* HM9, double* HN3, double* HNY3, double* HT9) {
  les_H_point(a, (const double (*)[LES_NAUX])da, (const double (*)[3])gu9, (const double (*)[3])gl9, sqrtg, p, (double (*)[3])HM9, HN3, HNY3, (double (*)[3])HT9);
}
void orc_les_aux_point(void* hh, const double* gl9, double sqrtg, const double* Bu, const double* prim, double* a26) {
  les_aux_point(((Handle*)hh)->par, (const double (*)[3])gl9, sqrtg, Bu, prim, a26);
}

void orc_eos_dp(void* hh, double rho, double eps, double ye, double* out3) { eos_dp(((Handle*)hh)->par, rho, eps, ye, out3[0], out3[1], out3[2]); }

// ---- AMR transfer operators (grids passed explicitly: n[3], ng)
static Grid mkgrid(const int* n, int ng) { return Grid{n[0], n[1], n[2], ng, 1.0, 1.0, 1.0}; }
void orc_prolong(const int* nc, int ngc, const double* Uc, const int* nf, int ngf, double* Uf, int nfields, const int* origin, const int* lo, const int* hi) {
  prolong(mkgrid(nc, ngc), Uc, mkgrid(nf, ngf), Uf, nfields, origin, lo, hi);
}
void orc_restrict(const int* nf, int ngf, const double* Uf, const int* nc, int ngc, double* Uc, int nfields, const int* origin) {
  restrict_copy(mkgrid(nf, ngf), Uf, mkgrid(nc, ngc), Uc, nfields, origin);
}
int orc_dense_weights(int scheme, double theta, int deriv, double* b4) { return dense_weights(scheme, theta, deriv, b4); }
void orc_dense_output(void* hh, int nfields, double* Uout, const double* U0, int scheme, const double* const* K, double theta, double dt, int deriv) {
  dense_output(((Handle*)hh)->grid, nfields, Uout, U0, scheme, K, theta, dt, deriv);
}
double orc_prolong_mid(const double* u, long s) { return prolong_mid(u, s); }

// ---- pointwise helpers for the pins
double orc_d1(const double* u, long s, double h) { return d1(u, s, h); }
double orc_d2(const double* u, long s, double h) { return d2(u, s, h); }
double orc_d11(const double* u, long s1, double h1, long s2, double h2) { return d11(u, s1, h1, s2, h2); }
double orc_dadv(const double* u, long s, double h, double beta) { return dadv(u, s, h, beta); }
double orc_dko(const double* u, long s, double h, double sigma) { return dko(u, s, h, sigma); }
double orc_mp5(double a, double b, double c, double d, double e, double alpha) { return mp5(a, b, c, d, e, alpha); }
double orc_weno5(double a, double b, double c, double d, double e, double eps) { return weno5(a, b, c, d, e, eps); }
void orc_eos(void* hh, double rho, double eps, double ye, double* out3) {
  const EosOut e = eos_from_rho_eps(((Handle*)hh)->par, rho, eps, ye);
  out3[0] = e.p; out3[1] = e.T; out3[2] = e.cs2;
}
double orc_eos_eps_from_T(void* hh, double rho, double T, double ye) { return eos_eps_from_T(((Handle*)hh)->par, rho, T, ye); }
int orc_con2prim_point(void* hh, const double* gt, double chi, double alpha, double* ucons, double* prim) {
  return con2prim_point(((Handle*)hh)->par, gt, chi, alpha, ucons, prim);
}
void orc_prim2con_point(const double* gl, const double* prim, const double* B, double* out5) {
  prim2con_point(gl, prim, B, out5[0], out5[1], out5 + 2);
}

}  // extern "C"
