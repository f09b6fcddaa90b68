// ORACLE (test infrastructure) — AMR transfer operators on a patch pair, Sec. IV B l.608-626 and the
// dense-output interpolator of Sec. III A, Eqs. (56)-(59) l.412-434. Plain definitions, written out.
//
// Geometry (refinement ratio 2, vertex-centred grids, l.620: "the points of the coarse grid also exist in the fine grid"): fine interior
// index a (any sign; ghosts have a < 0 or a >= n) sits at coarse position origin + a/2 along each axis; even a coincides with the coarse
// interior point origin + a/2, odd a is the midpoint between coarse points origin + (a-1)/2 and origin + (a+1)/2.
#include <cmath>
#include "orc.hpp"

namespace orc {

// Eq. (80), l.616: U_{i+1/2} = [150 (U_i + U_{i+1}) - 25 (U_{i-1} + U_{i+2}) + 3 (U_{i-2} + U_{i+3})] / 256, u points at U_i
double prolong_mid(const double* u, long s) {
  return (150.0 * (u[0] + u[s]) - 25.0 * (u[-s] + u[2 * s]) + 3.0 * (u[-2 * s] + u[3 * s])) / 256.0;
}

namespace {
// floor division by 2 and parity for either sign
inline int half_floor(int a) { return a >= 0 ? a / 2 : -((-a + 1) / 2); }
inline int parity(int a) { return a - 2 * half_floor(a); }

// 1-D weights of one fine point along one axis: coincident (1 weight at offset 0) or Eq. (80) (6 weights at offsets -2..3)
struct W1 { int n, off[6]; double w[6]; };
W1 weights(int par) {
  W1 r;
  if (par == 0) { r.n = 1; r.off[0] = 0; r.w[0] = 1.0; return r; }
  const double c[6] = {3.0 / 256.0, -25.0 / 256.0, 150.0 / 256.0, 150.0 / 256.0, -25.0 / 256.0, 3.0 / 256.0};
  r.n = 6;
  for (int m = 0; m < 6; ++m) { r.off[m] = m - 2; r.w[m] = c[m]; }
  return r;
}
}  // namespace

// Prolongation (l.608-620): every fine grid point of the index box [lo, hi) (ghosted fine array indices) is set from the coarse
// patch: the 1-D operator (copy / Eq. 80) applied along x, then y, then z (tensor product; reading R38: the paper prints the 1-D
// formula only).
void prolong(const Grid& gc, const double* Uc, const Grid& gf, double* Uf, int nfields, const int origin[3], const int lo[3], const int hi[3]) {
  const size_t nc = gc.npts(), nf = gf.npts();
  for (int f = 0; f < nfields; ++f)
    for (int K = lo[2]; K < hi[2]; ++K) for (int J = lo[1]; J < hi[1]; ++J) for (int I = lo[0]; I < hi[0]; ++I) {
      const int a[3] = {I - gf.ng, J - gf.ng, K - gf.ng};
      int c[3];
      W1 w[3];
      for (int d = 0; d < 3; ++d) { c[d] = origin[d] + half_floor(a[d]) + gc.ng; w[d] = weights(parity(a[d])); }
      double sz = 0.0;
      for (int n = 0; n < w[2].n; ++n) {
        double sy = 0.0;
        for (int m = 0; m < w[1].n; ++m) {
          double sx = 0.0;
          for (int l = 0; l < w[0].n; ++l)
            sx += w[0].w[l] * Uc[(size_t)f * nc + gc.idx(c[0] + w[0].off[l], c[1] + w[1].off[m], c[2] + w[2].off[n])];
          sy += w[1].w[m] * sx;
        }
        sz += w[2].w[n] * sy;
      }
      Uf[(size_t)f * nf + gf.idx(I, J, K)] = sz;
    }
}

// Restriction (l.626): direct copy of the fine interior points that coincide with coarse points
void restrict_copy(const Grid& gf, const double* Uf, const Grid& gc, double* Uc, int nfields, const int origin[3]) {
  const size_t nc = gc.npts(), nf = gf.npts();
  for (int f = 0; f < nfields; ++f)
    for (int k = 0; k < gf.nz; k += 2) for (int j = 0; j < gf.ny; j += 2) for (int i = 0; i < gf.nx; i += 2)
      Uc[(size_t)f * nc + gc.idx(origin[0] + i / 2 + gc.ng, origin[1] + j / 2 + gc.ng, origin[2] + k / 2 + gc.ng)] =
          Uf[(size_t)f * nf + gf.idx(i + gf.ng, j + gf.ng, k + gf.ng)];
}

// b_j(theta) of Eq. (58) (scheme 0: RK(4,4), third order) and Eq. (59) (scheme 1: SSP-RK(3,3), second order), or their deriv-th
// derivative with respect to theta (Eq. 57). Returns the number of stages.
int dense_weights(int scheme, double th, int deriv, double b[4]) {
  // polynomial coefficients p[j][m] of theta^m
  double p[4][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};
  int s;
  if (scheme == 0) {
    s = 4;
    p[0][1] = 1.0; p[0][2] = -3.0 / 2.0; p[0][3] = 2.0 / 3.0;     // b_1 = theta - 3/2 theta^2 + 2/3 theta^3
    p[1][2] = 1.0; p[1][3] = -2.0 / 3.0;                          // b_2 = b_3 = theta^2 - 2/3 theta^3
    p[2][2] = 1.0; p[2][3] = -2.0 / 3.0;
    p[3][2] = -1.0 / 2.0; p[3][3] = 2.0 / 3.0;                    // b_4 = -1/2 theta^2 + 2/3 theta^3
  } else {
    s = 3;
    p[0][1] = 1.0; p[0][2] = -5.0 / 6.0;                          // b_1 = theta - 5/6 theta^2
    p[1][2] = 1.0 / 6.0;                                          // b_2 = 1/6 theta^2
    p[2][2] = 4.0 / 6.0;                                          // b_3 = 4/6 theta^2
  }
  for (int j = 0; j < s; ++j) {
    double v = 0.0;
    for (int m = deriv; m < 4; ++m) {
      double c = p[j][m];
      for (int q = 0; q < deriv; ++q) c *= (double)(m - q);       // d^deriv/dtheta^deriv of theta^m
      v += c * std::pow(th, m - deriv);
    }
    b[j] = v;
  }
  return s;
}

// Eq. (56): U^{n+theta} = U^n + sum_j b_j(theta) k_j with k_j = dt K_j (K_j = F(U^(j)) as stored by the stage loop), interior points;
// deriv >= 1: Eq. (57), d^m U / dt^m = dt^-m sum_j k_j d^m b_j / dtheta^m (no U^n term).
void dense_output(const Grid& g, int nfields, double* Uout, const double* U0, int scheme, const double* const* K, double theta, double dt, int deriv) {
  double b[4];
  const int s = dense_weights(scheme, theta, deriv, b);
  const size_t n = g.npts();
  for (int f = 0; f < nfields; ++f)
    for (int k = g.ng; k < g.nz + g.ng; ++k) for (int j = g.ng; j < g.ny + g.ng; ++j) for (int i = g.ng; i < g.nx + g.ng; ++i) {
      const size_t p = (size_t)f * n + g.idx(i, j, k);
      double acc = 0.0;
      for (int m = 0; m < s; ++m) acc += b[m] * (dt * K[m][p]);
      Uout[p] = deriv == 0 ? U0[p] + acc : acc / std::pow(dt, deriv);
    }
}

}  // namespace orc
