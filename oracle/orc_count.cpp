// ORACLE (test infrastructure) — operation-counting build of the very same oracle sources.
//
// The seven oracle translation units are compiled unchanged with the token `double` replaced by a
// one-member wrapper whose arithmetic operators tick global counters. The resulting library
// (liboracle_count.so, same C entry points) therefore executes exactly the arithmetic of the
// oracle — with -ffp-contract=off no FMA can form — and reports the ALGORITHMIC floating-point
// operation count of whatever was run: the F_alg of SURVEY.md 8(d) / DESIGN.md "Measurement",
// used as the numerator of the FP64 roofline. Classes: add/sub, mul, div, sqrt, compare
// (<, >, ==, min, max), transcendental (pow, log, log10). fabs and unary minus are sign-bit
// operations and are not counted.
#include <algorithm>
#include <cfloat>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>

namespace orc_cnt {
unsigned long long n_add = 0, n_mul = 0, n_div = 0, n_sqrt = 0, n_cmp = 0, n_trans = 0;

struct Cnt {
  double v;
  Cnt() = default;
  Cnt(double x) : v(x) {}
  explicit operator int() const { return (int)v; }
  explicit operator long() const { return (long)v; }
  explicit operator unsigned char() const { return (unsigned char)v; }
  Cnt operator-() const { return Cnt(-v); }
  Cnt operator+() const { return *this; }
  Cnt& operator+=(Cnt b) { ++n_add; v += b.v; return *this; }
  Cnt& operator-=(Cnt b) { ++n_add; v -= b.v; return *this; }
  Cnt& operator*=(Cnt b) { ++n_mul; v *= b.v; return *this; }
  Cnt& operator/=(Cnt b) { ++n_div; v /= b.v; return *this; }
};
inline Cnt operator+(Cnt a, Cnt b) { ++n_add; return Cnt(a.v + b.v); }
inline Cnt operator-(Cnt a, Cnt b) { ++n_add; return Cnt(a.v - b.v); }
inline Cnt operator*(Cnt a, Cnt b) { ++n_mul; return Cnt(a.v * b.v); }
inline Cnt operator/(Cnt a, Cnt b) { ++n_div; return Cnt(a.v / b.v); }
inline bool operator<(Cnt a, Cnt b) { ++n_cmp; return a.v < b.v; }
inline bool operator>(Cnt a, Cnt b) { ++n_cmp; return a.v > b.v; }
inline bool operator<=(Cnt a, Cnt b) { ++n_cmp; return a.v <= b.v; }
inline bool operator>=(Cnt a, Cnt b) { ++n_cmp; return a.v >= b.v; }
inline bool operator==(Cnt a, Cnt b) { ++n_cmp; return a.v == b.v; }
inline bool operator!=(Cnt a, Cnt b) { ++n_cmp; return a.v != b.v; }
}  // namespace orc_cnt

namespace std {
inline orc_cnt::Cnt sqrt(orc_cnt::Cnt a) { ++orc_cnt::n_sqrt; return orc_cnt::Cnt(std::sqrt(a.v)); }
inline orc_cnt::Cnt fabs(orc_cnt::Cnt a) { return orc_cnt::Cnt(std::fabs(a.v)); }
inline orc_cnt::Cnt log(orc_cnt::Cnt a) { ++orc_cnt::n_trans; return orc_cnt::Cnt(std::log(a.v)); }
inline orc_cnt::Cnt log10(orc_cnt::Cnt a) { ++orc_cnt::n_trans; return orc_cnt::Cnt(std::log10(a.v)); }
inline orc_cnt::Cnt pow(orc_cnt::Cnt a, orc_cnt::Cnt b) { ++orc_cnt::n_trans; return orc_cnt::Cnt(std::pow(a.v, b.v)); }
inline orc_cnt::Cnt max(orc_cnt::Cnt a, orc_cnt::Cnt b) { ++orc_cnt::n_cmp; return a.v < b.v ? b : a; }
inline orc_cnt::Cnt min(orc_cnt::Cnt a, orc_cnt::Cnt b) { ++orc_cnt::n_cmp; return b.v < a.v ? b : a; }
inline orc_cnt::Cnt exp(orc_cnt::Cnt a) { ++orc_cnt::n_trans; return orc_cnt::Cnt(std::exp(a.v)); }
inline orc_cnt::Cnt tanh(orc_cnt::Cnt a) { ++orc_cnt::n_trans; return orc_cnt::Cnt(std::tanh(a.v)); }
}  // namespace std

using orc_cnt::Cnt;
#define double Cnt
#include "orc_stencil.cpp"
#include "orc_eos.cpp"
#include "orc_c2p.cpp"
#include "orc_ccz4.cpp"
#define SYM SYM_grmhd_unit
#include "orc_grmhd.cpp"
#undef SYM
#include "orc_rk.cpp"
#include "orc_m1.cpp"
#include "orc_m1_patch.cpp"
#include "orc_amr.cpp"
#define SYM SYM_les_unit
#include "orc_les.cpp"
#undef SYM
#include "orc_capi.cpp"
#undef double

extern "C" {
void orc_count_reset() { orc_cnt::n_add = orc_cnt::n_mul = orc_cnt::n_div = orc_cnt::n_sqrt = orc_cnt::n_cmp = orc_cnt::n_trans = 0; }
// out[6] = add/sub, mul, div, sqrt, compare/min/max, transcendental
void orc_count_get(unsigned long long* out) {
  out[0] = orc_cnt::n_add; out[1] = orc_cnt::n_mul; out[2] = orc_cnt::n_div;
  out[3] = orc_cnt::n_sqrt; out[4] = orc_cnt::n_cmp; out[5] = orc_cnt::n_trans;
}
}
