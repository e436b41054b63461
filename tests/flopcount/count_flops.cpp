// count_flops.cpp — re-derives the generator's hand-entered FLOPS tables (codegen/emit.py FLOPS, emit_orbit.py FL,
// emit_orbit5.py FL5) from csrc/hel_amp.cuh itself: the device routines are templates on the real type R, so they are
// instantiated here, on the host, with a scalar that COUNTS every +, -, *, / it executes (rule of SURVEY.md section 8(d):
// add = mul = div = sqrt = 1, hence fma = 2; unary minus and comparisons are free).  Prints one "name count" line per routine.
// Test infrastructure (tests/test_abi_and_host.py::test_flops_tables_match_the_device_routines); no CUDA needed.
#include <cmath>
#include <cstdio>

static long g_ops = 0;
struct Cnt {
  double v;
  Cnt() : v(0) {}
  Cnt(double x) : v(x) {}
  Cnt(int x) : v(x) {}
};
static inline Cnt operator+(Cnt a, Cnt b) { ++g_ops; return Cnt(a.v + b.v); }
static inline Cnt operator-(Cnt a, Cnt b) { ++g_ops; return Cnt(a.v - b.v); }
static inline Cnt operator*(Cnt a, Cnt b) { ++g_ops; return Cnt(a.v * b.v); }
static inline Cnt operator/(Cnt a, Cnt b) { ++g_ops; return Cnt(a.v / b.v); }
static inline Cnt operator-(Cnt a) { return Cnt(-a.v); }
static inline Cnt& operator+=(Cnt& a, Cnt b) { ++g_ops; a.v += b.v; return a; }
static inline Cnt& operator-=(Cnt& a, Cnt b) { ++g_ops; a.v -= b.v; return a; }
static inline Cnt& operator*=(Cnt& a, Cnt b) { ++g_ops; a.v *= b.v; return a; }
static inline bool operator>(Cnt a, Cnt b) { return a.v > b.v; }
static inline bool operator>=(Cnt a, Cnt b) { return a.v >= b.v; }
static inline bool operator==(Cnt a, Cnt b) { return a.v == b.v; }

#define ME_HOST_FLOP_COUNT 1
#include "hel_amp.cuh"

namespace me {
template <> inline Cnt rsqrt_<Cnt>(Cnt x) { g_ops += 2; return Cnt(1.0 / std::sqrt(x.v)); }
template <> inline Cnt sqrt_<Cnt>(Cnt x) { g_ops += 1; return Cnt(std::sqrt(x.v)); }
}  // namespace me

using namespace me;
typedef Cnt R;

static W4<R> some_w(double s) { return {R(0.3 + s), R(-0.7 * s), R(1.1), R(0.2 + s), R(-0.4), R(0.9 * s), R(0.5), R(-1.3 + s)}; }
static P4<R> some_p(double s) { return {R(5.0 + s), R(1.0 * s), R(-2.0), R(3.0 - s)}; }

#define COUNT(name, expr) do { g_ops = 0; auto r_ = (expr); (void)r_; std::printf("%s %ld\n", name, g_ops); } while (0)

int main() {
  const W4<R> a = some_w(0.1), b = some_w(0.7), c = some_w(-0.3);
  const P4<R> k1 = some_p(0.2), k2 = some_p(-0.6);
  const R m(173.0), iden(1e-3);
  COUNT("row_slash", row_slash(a, b));
  COUNT("slash_col", slash_col(a, b));
  COUNT("row_col", row_col(a, b));
  COUNT("wdot", wdot(a, b));
  COUNT("kdot", kdot(k1, a));
  COUNT("quark_step2", quark_step2(a, b, k1, m, iden));
  COUNT("col_step", col_step(a, k1, m, iden));
  COUNT("row_step", row_step(a, k1, m, iden));
  COUNT("v3_current", v3_current(a, b, k1, k2, iden));
  COUNT("v3_dual", v3_dual(a, b, k1, k2, iden));
  const V4Dots<R> d = v4_dots(a, b, c, iden);
  COUNT("v4_dots", v4_dots(a, b, c, iden));
  COUNT("v4_current", v4_current(0, d, a, b, c));
  COUNT("v4_current_1", v4_current(1, d, a, b, c));
  COUNT("v4_current_2", v4_current(2, d, a, b, c));
  COUNT("cx_comb", cx_comb(d.w12, a, d.w13, b));
  COUNT("bilinear", bilinear(a, b));
  COUNT("wadd", wadd(a, b));
  COUNT("wsub", wsub(a, b));
  // external states: the helicity-dependent part (the bases are per-event work, counted in `fixed`)
  const GluonBasis<R> gb = gluon_basis(some_p(0.3));
  COUNT("gluon_pol", gluon_pol_from(gb, R(1.0)));        // what the orbit kernels run; gluon_pol(): the sign s = +-1 is a compile-time constant
  COUNT("gluon_pol_in", gluon_pol(gb, R(1.0), false));
  COUNT("gluon_pol_out", gluon_pol(gb, R(-1.0), true));
  const SpinorBasis<R> sb = spinor_basis(some_p(0.4), m);
  COUNT("spinor_ubar_plus", spinor_ubar(sb, R(1.0)));
  COUNT("spinor_ubar_minus", spinor_ubar(sb, R(-1.0)));
  COUNT("spinor_v_plus", spinor_v(sb, R(1.0)));
  COUNT("spinor_v_minus", spinor_v(sb, R(-1.0)));
  COUNT("gluon_basis", gluon_basis(some_p(0.3)));
  COUNT("spinor_basis", spinor_basis(some_p(0.4), m));
  COUNT("padd", padd(k1, k2));
  COUNT("psub", psub(k1, k2));
  return 0;
}
