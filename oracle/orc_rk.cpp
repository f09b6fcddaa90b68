// ORACLE (test infrastructure) — ghost fill (readings R17), explicit Runge-Kutta
// combine (Eq. 53) and the per-stage driver of SURVEY call stack B.
#include <cstring>
#include <vector>
#include "orc.hpp"

namespace orc {

// bc[0..5] = {x-, x+, y-, y+, z-, z+}; 0 periodic wrap, 1 outflow (copy of the nearest interior value, R17).
// Done axis by axis (x, then y, then z) over the full extent of the other axes so edges and corners fill.
void fill_ghosts(const Grid& g, double* U, int nfields, const int bc[6]) {
  const size_t n = g.npts();
  const int M[3] = {g.mx(), g.my(), g.mz()};
  const int N[3] = {g.nx, g.ny, g.nz};
  const int ng = g.ng;
  for (int f = 0; f < nfields; ++f) {
    double* u = U + (size_t)f * n;
    for (int d = 0; d < 3; ++d) {
      int c[3];
      const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
      for (c[d2] = 0; c[d2] < M[d2]; ++c[d2]) for (c[d1] = 0; c[d1] < M[d1]; ++c[d1]) {
        for (int q = 0; q < ng; ++q) {
          int src[3] = {c[0], c[1], c[2]}, dst[3] = {c[0], c[1], c[2]};
          // low side: ghost index q
          dst[d] = q;
          src[d] = bc[2 * d] == 0 ? q + N[d] : ng;
          u[g.idx(dst[0], dst[1], dst[2])] = u[g.idx(src[0], src[1], src[2])];
          // high side: ghost index ng + N + q
          dst[d] = ng + N[d] + q;
          src[d] = bc[2 * d + 1] == 0 ? ng + q : ng + N[d] - 1;
          u[g.idx(dst[0], dst[1], dst[2])] = u[g.idx(src[0], src[1], src[2])];
        }
      }
    }
  }
}

// Uout = U0 + dt * sum_j coef[j] K_j on the interior (ghosts are refilled by fill_ghosts), Eq. (53)
void rk_combine(const Grid& g, int nfields, double* Uout, const double* U0, int nk,
                const double* const* K, const double* coef, double dt) {
  const size_t n = g.npts();
  for (int f = 0; f < nfields; ++f)
    for (int k = g.ng; k < g.nz + g.ng; ++k) for (int j = g.ng; j < g.ny + g.ng; ++j) for (int i = g.ng; i < g.nx + g.ng; ++i) {
      const size_t p = (size_t)f * n + g.idx(i, j, k);
      double s = 0.0;
      for (int m = 0; m < nk; ++m) s += coef[m] * K[m][p];
      Uout[p] = U0[p] + dt * s;
    }
}

// a_expl: row-major stages x stages (strictly lower triangular), w_expl: stages weights.
void evolve(const Params& par, const Grid& g, double* U, double* P, uint8_t* flags,
            const int bc[6], int stages, const double* a_expl, const double* w_expl,
            double dt, int n_steps) {
  const size_t nall = (size_t)NSTATE * g.npts();
  std::vector<double> U0(nall);
  std::vector<std::vector<double>> K(stages, std::vector<double>(nall, 0.0));
  std::vector<const double*> Kp(stages);
  for (int s = 0; s < stages; ++s) Kp[s] = K[s].data();
  for (int step = 0; step < n_steps; ++step) {
    // the state entering the step is made consistent first, so that U^n includes the con2prim resets
    fill_ghosts(g, U, NSTATE, bc);
    con2prim(par, g, U, P, flags);
    std::memcpy(U0.data(), U, nall * sizeof(double));
    for (int s = 0; s < stages; ++s) {
      if (s > 0) { fill_ghosts(g, U, NSTATE, bc); con2prim(par, g, U, P, flags); }
      rhs(par, g, U, P, K[s].data());
      if (s + 1 < stages) rk_combine(g, NSTATE, U, U0.data(), s + 1, Kp.data(), a_expl + (size_t)(s + 1) * stages, dt);
      else rk_combine(g, NSTATE, U, U0.data(), stages, Kp.data(), w_expl, dt);
    }
  }
  fill_ghosts(g, U, NSTATE, bc);
  con2prim(par, g, U, P, flags);
}

}  // namespace orc
