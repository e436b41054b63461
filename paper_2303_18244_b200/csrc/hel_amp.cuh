// =====================================================================================
// hel_amp.cuh — device wavefunction / vertex routines.
//
// External states, off-shell currents and amplitudes of the tree-level Feynman rules
// restated in DESIGN.md ("Readings" C1-C3): metric (+,-,-,-), chiral Dirac basis
//   gamma^0 = [[0,1],[1,0]],  gamma^i = [[0,s^i],[-s^i,0]],
// all gluon momenta counted INTO the vertex.  PAPER.md gives no formulas ("Feynman
// diagrams and helicity amplitudes"); these are the textbook rules.
//
// "Stripped" convention: every factor of i and of g_s is removed from the routines here.
// The generator (codegen/topology.py) folds the phases i^k into the Gaussian-integer colour
// coefficients c_{d,sigma} and the overall g_s^(2n) into the final normalisation, so all
// arithmetic below has real scalar coefficients only.
//
// Everything is a template on the real type R (double or float) and is force-inlined into
// the generated per-process kernels: one event per thread, no memory traffic in here.
// =====================================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace me {

#define ME_DEV __device__ __forceinline__
// compiler-only fence: memory operations are not moved across it (bounds load hoisting, hence register pressure)
#define ME_FENCE asm volatile("" ::: "memory")

template <typename R> struct P4 { R e, x, y, z; };            // real four-vector (E,px,py,pz)
template <typename R> struct Cx { R re, im; };
// four complex numbers: a Lorentz vector (contravariant 0..3) or a chiral-basis spinor
template <typename R> struct W4 { R r0, i0, r1, i1, r2, i2, r3, i3; };

template <typename R> ME_DEV R rsqrt_(R x);
template <> ME_DEV double rsqrt_<double>(double x) { return 1.0 / sqrt(x); }
template <> ME_DEV float rsqrt_<float>(float x) { return 1.0f / sqrtf(x); }
template <typename R> ME_DEV R sqrt_(R x);
template <> ME_DEV double sqrt_<double>(double x) { return sqrt(x); }
template <> ME_DEV float sqrt_<float>(float x) { return sqrtf(x); }

template <typename R> ME_DEV P4<R> padd(const P4<R>& a, const P4<R>& b) { return {a.e + b.e, a.x + b.x, a.y + b.y, a.z + b.z}; }
template <typename R> ME_DEV P4<R> psub(const P4<R>& a, const P4<R>& b) { return {a.e - b.e, a.x - b.x, a.y - b.y, a.z - b.z}; }
template <typename R> ME_DEV P4<R> pneg(const P4<R>& a) { return {-a.e, -a.x, -a.y, -a.z}; }
ME_DEV double pdot(const P4<double>& a, const P4<double>& b) { return a.e * b.e - a.x * b.x - a.y * b.y - a.z * b.z; }
template <typename R> ME_DEV P4<R> pcast(const P4<double>& a) { return {(R)a.e, (R)a.x, (R)a.y, (R)a.z}; }

#ifndef ME_HOST_FLOP_COUNT
// ------------------------------------------------------------------------------------
// Propagator denominators (helicity-independent, once per event, FP64 in every precision mode).  Without cuts some events
// have an invariant s_ij ~ 1e-6 s: (p_i + p_j)^2 formed in plain binary64 then carries a relative error eps * E^2 / s_ij, and
// the shortcut 2 p_i.p_j (which assumes exactly massless legs) differs from it by (p_i^2 + p_j^2) / s_ij, where p_i^2 ~ eps E^2 is
// the rounding of the input energy itself: both are 1e-10 effects on such events against north_star's 1e-11.  The invariants are
// therefore formed in double-double arithmetic (error-free products with FMA, compensated sums) from the binary64 inputs AS
// GIVEN, own squares p_i^2 and p_t^2 - m^2 included: K^2 and q^2 - m^2 are exact to rounding for the inputs the caller
// passed, which is what the oracle evaluated in long double computes.  ~1 kflop per event.
// ------------------------------------------------------------------------------------
struct DD { double hi, lo; };
ME_DEV DD dd_two_sum(double a, double b) {
  const double s = __dadd_rn(a, b), bb = __dadd_rn(s, -a);
  return {s, __dadd_rn(__dadd_rn(a, -__dadd_rn(s, -bb)), __dadd_rn(b, -bb))};
}
ME_DEV DD dd_two_prod(double a, double b) {
  const double p = __dmul_rn(a, b);
  return {p, __fma_rn(a, b, -p)};
}
ME_DEV DD dd_add(const DD& a, const DD& b) {
  const DD s = dd_two_sum(a.hi, b.hi);
  const double lo = __dadd_rn(__dadd_rn(a.lo, b.lo), s.lo);
  const double hi = __dadd_rn(s.hi, lo);
  return {hi, __dadd_rn(lo, -__dadd_rn(hi, -s.hi))};
}
ME_DEV DD dd_neg(const DD& a) { return {-a.hi, -a.lo}; }
ME_DEV DD dd_sub(const DD& a, const DD& b) { return dd_add(a, dd_neg(b)); }
ME_DEV DD dd_mul2(const DD& a) { return {2.0 * a.hi, 2.0 * a.lo}; }       // exact
ME_DEV double dd_value(const DD& a) { return __dadd_rn(a.hi, a.lo); }
// Minkowski product a.b of two binary64 four-vectors
ME_DEV DD dd_dot(const P4<double>& a, const P4<double>& b) {
  const DD t = dd_two_prod(a.e, b.e), x = dd_two_prod(a.x, b.x), y = dd_two_prod(a.y, b.y), z = dd_two_prod(a.z, b.z);
  return dd_sub(dd_sub(dd_sub(t, x), y), z);
}
// a.a - m^2
ME_DEV DD dd_offshell(const P4<double>& a, double m) { return dd_sub(dd_dot(a, a), dd_two_prod(m, m)); }
#endif

// ------------------------------------------------------------------------------------
// External gluons (step a3).  eps(p,lam) = (-lam e1 - i e2)/sqrt2 with real e1,e2 that do
// not depend on the helicity, so the basis is built once per event and a helicity flip is
// a sign.  pT = 0 branch: e1 = x^, e2 = sgn(pz) y^ (hit by both beams on every event).
// ------------------------------------------------------------------------------------
template <typename R> struct GluonBasis { R ax, ay, az, bx, by; };   // a = e1/sqrt2, b = e2/sqrt2

template <typename R> ME_DEV GluonBasis<R> gluon_basis(const P4<R>& p) {
  const R rs2 = (R)0.70710678118654752440;
  const R pt2 = p.x * p.x + p.y * p.y;
  GluonBasis<R> g;
  if (pt2 == (R)0) {
    g.ax = rs2; g.ay = 0; g.az = 0; g.bx = 0; g.by = p.z >= (R)0 ? rs2 : -rs2;
  } else {
    const R ipt = rsqrt_<R>(pt2), ipabs = rsqrt_<R>(pt2 + p.z * p.z);
    const R c = p.z * ipabs * ipt * rs2;
    g.ax = p.x * c; g.ay = p.y * c; g.az = -pt2 * ipt * ipabs * rs2;
    g.bx = -p.y * ipt * rs2; g.by = p.x * ipt * rs2;
  }
  return g;
}
// lam = +-1; outgoing gluons carry eps*
template <typename R> ME_DEV W4<R> gluon_pol(const GluonBasis<R>& g, R lam, bool outgoing) {
  W4<R> w;
  const R s = outgoing ? (R)1 : (R)-1;
  w.r0 = 0; w.i0 = 0;
  w.r1 = -lam * g.ax; w.i1 = s * g.bx;
  w.r2 = -lam * g.ay; w.i2 = s * g.by;
  w.r3 = -lam * g.az; w.i3 = 0;
  return w;
}

// ------------------------------------------------------------------------------------
// External fermions (step a3).  Two-spinors chi+ = (a, b+ic), chi- = (-b+ic, a) with
// a = N(|p|+pz), b = N px, c = N py, N = 1/sqrt(2|p|(|p|+pz)); |p|+pz = 0: chi+ = (0,1),
// chi- = (-1,0).  wp = sqrt(E+|p|), wm = sqrt(E-|p|) = m/wp (exactly 0 for m = 0).
// ------------------------------------------------------------------------------------
template <typename R> struct SpinorBasis { R a, b, c, wp, wm; };

template <typename R> ME_DEV SpinorBasis<R> spinor_basis(const P4<R>& p, R m) {
  SpinorBasis<R> s;
  const R pt2 = p.x * p.x + p.y * p.y;
  R pabs;
  if (m == (R)0) { pabs = p.e; s.wp = sqrt_<R>((R)2 * p.e); s.wm = 0; }
  else { pabs = sqrt_<R>(pt2 + p.z * p.z); s.wp = sqrt_<R>(p.e + pabs); s.wm = m / s.wp; }
  const R ppz = p.z >= (R)0 ? pabs + p.z : pt2 / (pabs - p.z);
  if (ppz == (R)0) { s.a = 0; s.b = 1; s.c = 0; }
  else { const R N = rsqrt_<R>((R)2 * pabs * ppz); s.a = N * ppz; s.b = N * p.x; s.c = N * p.y; }
  return s;
}
// ubar(p,lam) = u^dagger gamma^0 (row spinor) — outgoing fermion
template <typename R> ME_DEV W4<R> spinor_ubar(const SpinorBasis<R>& s, R lam) {
  W4<R> w;
  if (lam > (R)0) {   // chi+^* = (a, b - ic)
    w.r0 = s.wp * s.a; w.i0 = 0; w.r1 = s.wp * s.b; w.i1 = -s.wp * s.c;
    w.r2 = s.wm * s.a; w.i2 = 0; w.r3 = s.wm * s.b; w.i3 = -s.wm * s.c;
  } else {            // chi-^* = (-b - ic, a)
    w.r0 = -s.wm * s.b; w.i0 = -s.wm * s.c; w.r1 = s.wm * s.a; w.i1 = 0;
    w.r2 = -s.wp * s.b; w.i2 = -s.wp * s.c; w.r3 = s.wp * s.a; w.i3 = 0;
  }
  return w;
}
// v(p,lam) (column spinor) — outgoing antifermion of physical helicity lam
template <typename R> ME_DEV W4<R> spinor_v(const SpinorBasis<R>& s, R lam) {
  W4<R> w;
  if (lam > (R)0) {   // (-wp chi-, wm chi-)
    w.r0 = s.wp * s.b; w.i0 = -s.wp * s.c; w.r1 = -s.wp * s.a; w.i1 = 0;
    w.r2 = -s.wm * s.b; w.i2 = s.wm * s.c; w.r3 = s.wm * s.a; w.i3 = 0;
  } else {            // (wm chi+, -wp chi+)
    w.r0 = s.wm * s.a; w.i0 = 0; w.r1 = s.wm * s.b; w.i1 = s.wm * s.c;
    w.r2 = -s.wp * s.a; w.i2 = 0; w.r3 = -s.wp * s.b; w.i3 = -s.wp * s.c;
  }
  return w;
}
// u(p,lam) (column spinor) — incoming fermion
template <typename R> ME_DEV W4<R> spinor_u(const SpinorBasis<R>& s, R lam) {
  W4<R> w;
  if (lam > (R)0) {   // (wm chi+, wp chi+)
    w.r0 = s.wm * s.a; w.i0 = 0; w.r1 = s.wm * s.b; w.i1 = s.wm * s.c;
    w.r2 = s.wp * s.a; w.i2 = 0; w.r3 = s.wp * s.b; w.i3 = s.wp * s.c;
  } else {            // (wp chi-, wm chi-)
    w.r0 = -s.wp * s.b; w.i0 = s.wp * s.c; w.r1 = s.wp * s.a; w.i1 = 0;
    w.r2 = -s.wm * s.b; w.i2 = s.wm * s.c; w.r3 = s.wm * s.a; w.i3 = 0;
  }
  return w;
}
// psibar = psi^dagger gamma^0: swap the chirality blocks and conjugate
template <typename R> ME_DEV W4<R> dirac_bar(const W4<R>& s) {
  return {s.r2, -s.i2, s.r3, -s.i3, s.r0, -s.i0, s.r1, -s.i1};
}

// ------------------------------------------------------------------------------------
// Dirac algebra.  V-slash = [[0, S],[Sb, 0]],  S = [[A,-C],[-D,B]],  Sb = [[B,C],[D,A]],
// A = V0-V3, B = V0+V3, C = V1-iV2, D = V1+iV2.
// ------------------------------------------------------------------------------------
#define ME_CMUL_RE(ar, ai, br, bi) ((ar) * (br) - (ai) * (bi))
#define ME_CMUL_IM(ar, ai, br, bi) ((ar) * (bi) + (ai) * (br))

// All sums of products below are written as FLAT left-to-right chains (no parenthesised partial sums) so
// that nvcc contracts them into one multiply followed by fused multiply-adds: the FP64 pipe issues one
// instruction per term instead of a mul + an add (profiles/r1_*: only 38 % of FP64 instructions were DFMA).
// row spinor times V-slash (complex V)
template <typename R> ME_DEV W4<R> row_slash(const W4<R>& r, const W4<R>& V) {
  const R Ar = V.r0 - V.r3, Ai = V.i0 - V.i3, Br = V.r0 + V.r3, Bi = V.i0 + V.i3;
  const R Cr = V.r1 + V.i2, Ci = V.i1 - V.r2, Dr = V.r1 - V.i2, Di = V.i1 + V.r2;
  W4<R> o;
  o.r2 = r.r0 * Ar - r.i0 * Ai - r.r1 * Dr + r.i1 * Di;
  o.i2 = r.r0 * Ai + r.i0 * Ar - r.r1 * Di - r.i1 * Dr;
  o.r3 = r.r1 * Br - r.i1 * Bi - r.r0 * Cr + r.i0 * Ci;
  o.i3 = r.r1 * Bi + r.i1 * Br - r.r0 * Ci - r.i0 * Cr;
  o.r0 = r.r2 * Br - r.i2 * Bi + r.r3 * Dr - r.i3 * Di;
  o.i0 = r.r2 * Bi + r.i2 * Br + r.r3 * Di + r.i3 * Dr;
  o.r1 = r.r2 * Cr - r.i2 * Ci + r.r3 * Ar - r.i3 * Ai;
  o.i1 = r.r2 * Ci + r.i2 * Cr + r.r3 * Ai + r.i3 * Ar;
  return o;
}
// V-slash (complex V) times column spinor
template <typename R> ME_DEV W4<R> slash_col(const W4<R>& V, const W4<R>& c) {
  const R Ar = V.r0 - V.r3, Ai = V.i0 - V.i3, Br = V.r0 + V.r3, Bi = V.i0 + V.i3;
  const R Cr = V.r1 + V.i2, Ci = V.i1 - V.r2, Dr = V.r1 - V.i2, Di = V.i1 + V.r2;
  W4<R> o;
  o.r0 = Ar * c.r2 - Ai * c.i2 - Cr * c.r3 + Ci * c.i3;
  o.i0 = Ar * c.i2 + Ai * c.r2 - Cr * c.i3 - Ci * c.r3;
  o.r1 = Br * c.r3 - Bi * c.i3 - Dr * c.r2 + Di * c.i2;
  o.i1 = Br * c.i3 + Bi * c.r3 - Dr * c.i2 - Di * c.r2;
  o.r2 = Br * c.r0 - Bi * c.i0 + Cr * c.r1 - Ci * c.i1;
  o.i2 = Br * c.i0 + Bi * c.r0 + Cr * c.i1 + Ci * c.r1;
  o.r3 = Dr * c.r0 - Di * c.i0 + Ar * c.r1 - Ai * c.i1;
  o.i3 = Dr * c.i0 + Di * c.r0 + Ar * c.i1 + Ai * c.r1;
  return o;
}
// row . column
template <typename R> ME_DEV Cx<R> row_col(const W4<R>& r, const W4<R>& c) {
  Cx<R> o;
  o.re = r.r0 * c.r0 - r.i0 * c.i0 + r.r1 * c.r1 - r.i1 * c.i1 + r.r2 * c.r2 - r.i2 * c.i2 + r.r3 * c.r3 - r.i3 * c.i3;
  o.im = r.r0 * c.i0 + r.i0 * c.r0 + r.r1 * c.i1 + r.i1 * c.r1 + r.r2 * c.i2 + r.i2 * c.r2 + r.r3 * c.i3 + r.i3 * c.r3;
  return o;
}
// Minkowski products
template <typename R> ME_DEV Cx<R> wdot(const W4<R>& a, const W4<R>& b) {
  Cx<R> o;
  o.re = a.r0 * b.r0 - a.i0 * b.i0 - a.r1 * b.r1 + a.i1 * b.i1 - a.r2 * b.r2 + a.i2 * b.i2 - a.r3 * b.r3 + a.i3 * b.i3;
  o.im = a.r0 * b.i0 + a.i0 * b.r0 - a.r1 * b.i1 - a.i1 * b.r1 - a.r2 * b.i2 - a.i2 * b.r2 - a.r3 * b.i3 - a.i3 * b.r3;
  return o;
}
template <typename R> ME_DEV Cx<R> kdot(const P4<R>& k, const W4<R>& w) {
  return {k.e * w.r0 - k.x * w.r1 - k.y * w.r2 - k.z * w.r3, k.e * w.i0 - k.x * w.i1 - k.y * w.i2 - k.z * w.i3};
}

// ------------------------------------------------------------------------------------
// Off-shell currents (step a4), stripped of i and g_s.
// ------------------------------------------------------------------------------------
// Quark line grown from the outgoing t (row spinor): psibar' = psibar V-slash (q-slash + m) * iden,
// q = fermion-flow momentum of the new propagator, iden = 1/(q^2 - m^2).
template <typename R> ME_DEV W4<R> quark_step2(const W4<R>& psibar, const W4<R>& V, const P4<R>& q, R m, R iden);
template <typename R> ME_DEV W4<R> quark_step(const W4<R>& psibar, const W4<R>& V, const P4<R>& q, R m, R iden) {
  return quark_step2(psibar, V, q, m, iden);
}
// Three-gluon vertex current, legs 1,2 with incoming momenta k1,k2, open leg momentum -(k1+k2):
//   W = [ (W1.W2)(k1-k2) + ((k1+2k2).W1) W2 - ((2k1+k2).W2) W1 ] * ik2 ,  ik2 = 1/(k1+k2)^2
template <typename R> ME_DEV W4<R> v3_current(const W4<R>& W1, const W4<R>& W2, const P4<R>& k1, const P4<R>& k2, R ik2) {
  Cx<R> w12 = wdot(W1, W2);
  const P4<R> ka = {k1.e + (R)2 * k2.e, k1.x + (R)2 * k2.x, k1.y + (R)2 * k2.y, k1.z + (R)2 * k2.z};
  const P4<R> kb = {(R)2 * k1.e + k2.e, (R)2 * k1.x + k2.x, (R)2 * k1.y + k2.y, (R)2 * k1.z + k2.z};
  Cx<R> a = kdot(ka, W1), b = kdot(kb, W2);
  w12.re *= ik2; w12.im *= ik2; a.re *= ik2; a.im *= ik2; b.re *= ik2; b.im *= ik2;
  const P4<R> d = psub(k1, k2);
  W4<R> o;
  o.r0 = w12.re * d.e + a.re * W2.r0 - a.im * W2.i0 - b.re * W1.r0 + b.im * W1.i0;
  o.i0 = w12.im * d.e + a.re * W2.i0 + a.im * W2.r0 - b.re * W1.i0 - b.im * W1.r0;
  o.r1 = w12.re * d.x + a.re * W2.r1 - a.im * W2.i1 - b.re * W1.r1 + b.im * W1.i1;
  o.i1 = w12.im * d.x + a.re * W2.i1 + a.im * W2.r1 - b.re * W1.i1 - b.im * W1.r1;
  o.r2 = w12.re * d.y + a.re * W2.r2 - a.im * W2.i2 - b.re * W1.r2 + b.im * W1.i2;
  o.i2 = w12.im * d.y + a.re * W2.i2 + a.im * W2.r2 - b.re * W1.i2 - b.im * W1.r2;
  o.r3 = w12.re * d.z + a.re * W2.r3 - a.im * W2.i3 - b.re * W1.r3 + b.im * W1.i3;
  o.i3 = w12.im * d.z + a.re * W2.i3 + a.im * W2.r3 - b.re * W1.i3 - b.im * W1.r3;
  return o;
}
// Four-gluon vertex: the three kinematic structures share the products W1.W2, W1.W3, W2.W3
//   s0 = (W1.W3) W2 - (W2.W3) W1     [f^{abe}f^{cde}]
//   s1 = (W1.W2) W3 - (W2.W3) W1     [f^{ace}f^{bde}]
//   s2 = (W1.W2) W3 - (W1.W3) W2     [f^{ade}f^{bce}]      each times ik2
template <typename R> struct V4Dots { Cx<R> w12, w13, w23; };
template <typename R> ME_DEV V4Dots<R> v4_dots(const W4<R>& W1, const W4<R>& W2, const W4<R>& W3, R ik2) {
  V4Dots<R> d; d.w12 = wdot(W1, W2); d.w13 = wdot(W1, W3); d.w23 = wdot(W2, W3);
  d.w12.re *= ik2; d.w12.im *= ik2; d.w13.re *= ik2; d.w13.im *= ik2; d.w23.re *= ik2; d.w23.im *= ik2;
  return d;
}
template <typename R> ME_DEV W4<R> cx_comb(const Cx<R>& a, const W4<R>& X, const Cx<R>& b, const W4<R>& Y) {   // a X - b Y
  W4<R> o;
  o.r0 = a.re * X.r0 - a.im * X.i0 - b.re * Y.r0 + b.im * Y.i0;
  o.i0 = a.re * X.i0 + a.im * X.r0 - b.re * Y.i0 - b.im * Y.r0;
  o.r1 = a.re * X.r1 - a.im * X.i1 - b.re * Y.r1 + b.im * Y.i1;
  o.i1 = a.re * X.i1 + a.im * X.r1 - b.re * Y.i1 - b.im * Y.r1;
  o.r2 = a.re * X.r2 - a.im * X.i2 - b.re * Y.r2 + b.im * Y.i2;
  o.i2 = a.re * X.i2 + a.im * X.r2 - b.re * Y.i2 - b.im * Y.r2;
  o.r3 = a.re * X.r3 - a.im * X.i3 - b.re * Y.r3 + b.im * Y.i3;
  o.i3 = a.re * X.i3 + a.im * X.r3 - b.re * Y.i3 - b.im * Y.r3;
  return o;
}
template <typename R> ME_DEV W4<R> v4_current(int k, const V4Dots<R>& d, const W4<R>& W1, const W4<R>& W2, const W4<R>& W3) {
  if (k == 0) return cx_comb(d.w13, W2, d.w23, W1);
  if (k == 1) return cx_comb(d.w12, W3, d.w23, W1);
  return cx_comb(d.w12, W3, d.w13, W2);
}
// fermion bilinear  J^mu = row gamma^mu col  (contravariant), used to close a gluon tree on the bare line:
//   row Vslash col = V . J
template <typename R> ME_DEV W4<R> bilinear(const W4<R>& r, const W4<R>& c) {
  // gamma^0: blocks [[0,1],[1,0]]; gamma^i: [[0,s^i],[-s^i,0]]
  // upper-right block couples (r0,r1) with (c2,c3); lower-left couples (r2,r3) with (c0,c1)
  const R u00r = ME_CMUL_RE(r.r0, r.i0, c.r2, c.i2), u00i = ME_CMUL_IM(r.r0, r.i0, c.r2, c.i2);
  const R u01r = ME_CMUL_RE(r.r0, r.i0, c.r3, c.i3), u01i = ME_CMUL_IM(r.r0, r.i0, c.r3, c.i3);
  const R u10r = ME_CMUL_RE(r.r1, r.i1, c.r2, c.i2), u10i = ME_CMUL_IM(r.r1, r.i1, c.r2, c.i2);
  const R u11r = ME_CMUL_RE(r.r1, r.i1, c.r3, c.i3), u11i = ME_CMUL_IM(r.r1, r.i1, c.r3, c.i3);
  const R l00r = ME_CMUL_RE(r.r2, r.i2, c.r0, c.i0), l00i = ME_CMUL_IM(r.r2, r.i2, c.r0, c.i0);
  const R l01r = ME_CMUL_RE(r.r2, r.i2, c.r1, c.i1), l01i = ME_CMUL_IM(r.r2, r.i2, c.r1, c.i1);
  const R l10r = ME_CMUL_RE(r.r3, r.i3, c.r0, c.i0), l10i = ME_CMUL_IM(r.r3, r.i3, c.r0, c.i0);
  const R l11r = ME_CMUL_RE(r.r3, r.i3, c.r1, c.i1), l11i = ME_CMUL_IM(r.r3, r.i3, c.r1, c.i1);
  W4<R> J;
  // J^0 = u00+u11 + l00+l11
  J.r0 = u00r + u11r + l00r + l11r; J.i0 = u00i + u11i + l00i + l11i;
  // J^1: sigma^1 = [[0,1],[1,0]] : (u01+u10) - (l01+l10)
  J.r1 = u01r + u10r - l01r - l10r; J.i1 = u01i + u10i - l01i - l10i;
  // J^2: sigma^2 = [[0,-i],[i,0]] : -i u01 + i u10 - (-i l01 + i l10)
  J.r2 = u01i - u10i - l01i + l10i; J.i2 = -u01r + u10r + l01r - l10r;
  // J^3: sigma^3 = diag(1,-1): (u00-u11) - (l00-l11)
  J.r3 = u00r - u11r - l00r + l11r; J.i3 = u00i - u11i - l00i + l11i;
  return J;
}

}  // namespace me

#ifndef ME_HOST_FLOP_COUNT   // tests/flopcount instantiates the arithmetic routines on the host; storage helpers are CUDA-only
// ------------------------------------------------------------------------------------
// Per-thread shared-memory slots.  Slots are stored in PAIRS: slot s of thread t is element
//     2 * ((s >> 1) * ME_SM_STRIDE + t) + (s & 1)        (ME_SM_STRIDE = threads per CTA)
// of an R array, so two consecutive slots (an even one and its successor: re/im of a complex number,
// half of a four-vector) are one 16-byte (FP64) / 8-byte (FP32) access per thread, conflict-free
// across the warp, and a complex current is 4 loads instead of 8.  `sm` below is the R pointer already
// offset by 2*threadIdx.x; ME_EO(s) is the element offset of slot s.  Vector types start on even slots.
// ------------------------------------------------------------------------------------
#ifndef ME_SM_STRIDE
#define ME_SM_STRIDE 128
#endif
#define ME_EO(s) ((((s) >> 1) * 2 * ME_SM_STRIDE) + ((s) & 1))
namespace me {
template <typename R> struct Pair2;
template <> struct Pair2<double> { typedef double2 T; };
template <> struct Pair2<float> { typedef float2 T; };
// pointer-based forms: p = sm + ME_EO(even slot)
template <typename R> ME_DEV W4<R> ldw(const R* p) {
  typedef typename Pair2<R>::T R2;
  const R2* q = reinterpret_cast<const R2*>(p);
  const R2 a = q[0], b = q[ME_SM_STRIDE], c = q[2 * ME_SM_STRIDE], d = q[3 * ME_SM_STRIDE];
  return {a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y};
}
template <typename R> ME_DEV void stw(R* p, const W4<R>& w) {
  typedef typename Pair2<R>::T R2;
  R2* q = reinterpret_cast<R2*>(p);
  R2 a, b, c, d; a.x = w.r0; a.y = w.i0; b.x = w.r1; b.y = w.i1; c.x = w.r2; c.y = w.i2; d.x = w.r3; d.y = w.i3;
  q[0] = a; q[ME_SM_STRIDE] = b; q[2 * ME_SM_STRIDE] = c; q[3 * ME_SM_STRIDE] = d;
}
template <typename R> ME_DEV P4<R> ldp(const R* p) {
  typedef typename Pair2<R>::T R2;
  const R2* q = reinterpret_cast<const R2*>(p);
  const R2 a = q[0], b = q[ME_SM_STRIDE];
  return {a.x, a.y, b.x, b.y};
}
template <typename R> ME_DEV void stp(R* p, const P4<R>& v) {
  typedef typename Pair2<R>::T R2;
  R2* q = reinterpret_cast<R2*>(p);
  R2 a, b; a.x = v.e; a.y = v.x; b.x = v.y; b.y = v.z;
  q[0] = a; q[ME_SM_STRIDE] = b;
}
// five reals (polarisation basis, spinor basis): two pairs + one single (the sixth slot is free for a scalar)
template <typename R> ME_DEV void ld5(const R* p, R& v0, R& v1, R& v2, R& v3, R& v4) {
  typedef typename Pair2<R>::T R2;
  const R2* q = reinterpret_cast<const R2*>(p);
  const R2 a = q[0], b = q[ME_SM_STRIDE];
  v0 = a.x; v1 = a.y; v2 = b.x; v3 = b.y; v4 = p[4 * ME_SM_STRIDE];
}
template <typename R> ME_DEV void st5(R* p, R v0, R v1, R v2, R v3, R v4) {
  typedef typename Pair2<R>::T R2;
  R2* q = reinterpret_cast<R2*>(p);
  R2 a, b; a.x = v0; a.y = v1; b.x = v2; b.y = v3;
  q[0] = a; q[ME_SM_STRIDE] = b; p[4 * ME_SM_STRIDE] = v4;
}
template <typename R> ME_DEV GluonBasis<R> ldgb(const R* p) { GluonBasis<R> g; ld5<R>(p, g.ax, g.ay, g.az, g.bx, g.by); return g; }
template <typename R> ME_DEV void stgb(R* p, const GluonBasis<R>& g) { st5<R>(p, g.ax, g.ay, g.az, g.bx, g.by); }
template <typename R> ME_DEV SpinorBasis<R> ldsb(const R* p) { SpinorBasis<R> g; ld5<R>(p, g.a, g.b, g.c, g.wp, g.wm); return g; }
template <typename R> ME_DEV void stsb(R* p, const SpinorBasis<R>& g) { st5<R>(p, g.a, g.b, g.c, g.wp, g.wm); }
// slot-index forms (static slot numbers)
template <typename R> ME_DEV W4<R> ldw(const R* sm, int s) { return ldw<R>(sm + ME_EO(s)); }
template <typename R> ME_DEV void stw(R* sm, int s, const W4<R>& w) { stw<R>(sm + ME_EO(s), w); }
template <typename R> ME_DEV P4<R> ldp(const R* sm, int s) { return ldp<R>(sm + ME_EO(s)); }
template <typename R> ME_DEV void stp(R* sm, int s, const P4<R>& v) { stp<R>(sm + ME_EO(s), v); }
template <typename R> ME_DEV GluonBasis<R> ldgb(const R* sm, int s) { return ldgb<R>(sm + ME_EO(s)); }
template <typename R> ME_DEV void stgb(R* sm, int s, const GluonBasis<R>& g) { stgb<R>(sm + ME_EO(s), g); }
template <typename R> ME_DEV SpinorBasis<R> ldsb(const R* sm, int s) { return ldsb<R>(sm + ME_EO(s)); }
template <typename R> ME_DEV void stsb(R* sm, int s, const SpinorBasis<R>& g) { stsb<R>(sm + ME_EO(s), g); }
template <typename R> ME_DEV void cset(R* p, R re, R im) {
  typedef typename Pair2<R>::T R2;
  R2 v; v.x = re; v.y = im; *reinterpret_cast<R2*>(p) = v;
}
template <typename R> ME_DEV void cget(const R* p, R& re, R& im) {
  typedef typename Pair2<R>::T R2;
  const R2 v = *reinterpret_cast<const R2*>(p); re = v.x; im = v.y;
}
// complex accumulator in a slot pair: one vector load, one vector store
template <typename R> ME_DEV void cacc(R* p, R dre, R dim) {
  typedef typename Pair2<R>::T R2;
  R2* q = reinterpret_cast<R2*>(p);
  R2 v = *q; v.x += dre; v.y += dim; *q = v;
}
}  // namespace me

// ------------------------------------------------------------------------------------
// Tensor memory as a per-thread scratchpad (FP64 kernels of g g -> t t~ g g).  The diagram kernels have no matrix
// product to give to tcgen05.mma, but with 226 FP64 slots per thread shared memory admits only ONE 128-thread CTA per SM
// (one warp per scheduler: every shared-memory and FP64 latency is exposed).  The 256 KB of TMEM are 128 lanes x 512
// 32-bit columns; a thread that owns lane (warp % 4) * 32 + laneid can keep 128 more FP64 slots in 256 columns of it,
// reached with tcgen05.ld / tcgen05.st (.32x32b: lane i of the warp <-> TMEM lane base + i, the column offset is
// warp-uniform, which table-driven lockstep code satisfies by construction).  Two CTAs per SM then fit: 98 slots in
// shared memory + 128 in TMEM each.  Slot s >= ME_TM_SLOT0 lives in TMEM at column 2 * (s - ME_TM_SLOT0); the emitter
// keeps passing the shared-memory element offset of the slot (what the FP32 kernel uses) and ME_TM_COL converts it.
// Loads are split into issue / get so that several are in flight before the one tcgen05.wait::ld; the loaded registers
// are operands of the wait so that no use can be scheduled above it.
// ------------------------------------------------------------------------------------
#ifndef ME_TM_SLOT0
#define ME_TM_SLOT0 0
#endif
// (the element offset of even slot s is ME_SM_STRIDE * s; ME_SM_STRIDE is a power of two: 128 threads per CTA, or 256 in the kernels
// whose two groups of four warps share the TMEM lanes and take half of the columns each)
// columns per slot: 2 for FP64, 1 for FP32
#define ME_TM_COL(R, off) (((uint32_t)(off) * (uint32_t)(sizeof(R) / 4)) / (uint32_t)ME_SM_STRIDE - (uint32_t)((sizeof(R) / 4) * ME_TM_SLOT0))
namespace me {
ME_DEV void tm_ld16(uint32_t (&r)[16], uint32_t a) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                 "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(a));
}
ME_DEV void tm_wait_ld16(uint32_t (&r)[16]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]), "+r"(r[8]), "+r"(r[9]),
                 "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15]));
}
ME_DEV void tm_ld8(uint32_t (&r)[8], uint32_t a) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(a));
}
ME_DEV void tm_wait_ld8(uint32_t (&r)[8]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]));
}
ME_DEV void tm_ld4(uint32_t (&r)[4], uint32_t a) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(a));
}
ME_DEV void tm_wait_ld4(uint32_t (&r)[4]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]));
}
ME_DEV void tm_ld2(uint32_t (&r)[2], uint32_t a) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "r"(a));
}
ME_DEV void tm_wait_ld2(uint32_t (&r)[2]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(r[0]), "+r"(r[1]));
}
ME_DEV void tm_st16(uint32_t a, const uint32_t (&r)[16]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(a),
               "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]),
               "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]));
}
ME_DEV void tm_st8(uint32_t a, const uint32_t (&r)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(a),
               "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]));
}
ME_DEV void tm_st4(uint32_t a, uint32_t r0, uint32_t r1, uint32_t r2, uint32_t r3) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(r0), "r"(r1), "r"(r2), "r"(r3));
}
ME_DEV void tm_st2(uint32_t a, uint32_t r0, uint32_t r1) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(a), "r"(r0), "r"(r1));
}
// a 4-vector load in flight: from shared memory it is complete at issue; from TMEM it is 16 (FP64) or 8 (FP32) raw registers until xldw_get
template <typename R, bool TM> struct XW { W4<R> w; };
template <> struct XW<double, true> { uint32_t r[16]; };
template <> struct XW<float, true> { uint32_t r[8]; };
template <typename R, bool TM> struct XC { R re, im; };
template <> struct XC<double, true> { uint32_t r[4]; };
template <> struct XC<float, true> { uint32_t r[2]; };
template <typename R, bool TM> ME_DEV void xldw_issue(XW<R, TM>& x, const R* sm, uint32_t tm, int off) {
  if constexpr (TM && sizeof(R) == 8) tm_ld16(x.r, tm + ME_TM_COL(R, off));
  else if constexpr (TM) tm_ld8(x.r, tm + ME_TM_COL(R, off));
  else x.w = ldw<R>(sm + off);
}
template <typename R, bool TM> ME_DEV W4<R> xldw_get(XW<R, TM>& x) {
  if constexpr (TM && sizeof(R) == 8) {
    tm_wait_ld16(x.r);
    return {__hiloint2double(x.r[1], x.r[0]), __hiloint2double(x.r[3], x.r[2]), __hiloint2double(x.r[5], x.r[4]), __hiloint2double(x.r[7], x.r[6]),
            __hiloint2double(x.r[9], x.r[8]), __hiloint2double(x.r[11], x.r[10]), __hiloint2double(x.r[13], x.r[12]), __hiloint2double(x.r[15], x.r[14])};
  } else if constexpr (TM) {
    tm_wait_ld8(x.r);
    return {__uint_as_float(x.r[0]), __uint_as_float(x.r[1]), __uint_as_float(x.r[2]), __uint_as_float(x.r[3]),
            __uint_as_float(x.r[4]), __uint_as_float(x.r[5]), __uint_as_float(x.r[6]), __uint_as_float(x.r[7])};
  } else {
    return x.w;
  }
}
template <typename R, bool TM> ME_DEV void xstw(R* sm, uint32_t tm, int off, const W4<R>& w) {
  if constexpr (TM && sizeof(R) == 8) {
    const double v[8] = {w.r0, w.i0, w.r1, w.i1, w.r2, w.i2, w.r3, w.i3};
    uint32_t r[16];
#pragma unroll
    for (int k = 0; k < 8; ++k) { r[2 * k] = (uint32_t)__double2loint(v[k]); r[2 * k + 1] = (uint32_t)__double2hiint(v[k]); }
    tm_st16(tm + ME_TM_COL(R, off), r);
  } else if constexpr (TM) {
    const uint32_t r[8] = {__float_as_uint(w.r0), __float_as_uint(w.i0), __float_as_uint(w.r1), __float_as_uint(w.i1),
                           __float_as_uint(w.r2), __float_as_uint(w.i2), __float_as_uint(w.r3), __float_as_uint(w.i3)};
    tm_st8(tm + ME_TM_COL(R, off), r);
  } else {
    stw<R>(sm + off, w);
  }
}
template <typename R, bool TM> ME_DEV void xcget_issue(XC<R, TM>& x, const R* sm, uint32_t tm, int off) {
  if constexpr (TM && sizeof(R) == 8) tm_ld4(x.r, tm + ME_TM_COL(R, off));
  else if constexpr (TM) tm_ld2(x.r, tm + ME_TM_COL(R, off));
  else cget<R>(sm + off, x.re, x.im);
}
template <typename R, bool TM> ME_DEV void xcget_get(XC<R, TM>& x, R& re, R& im) {
  if constexpr (TM && sizeof(R) == 8) {
    tm_wait_ld4(x.r);
    re = __hiloint2double(x.r[1], x.r[0]); im = __hiloint2double(x.r[3], x.r[2]);
  } else if constexpr (TM) {
    tm_wait_ld2(x.r);
    re = __uint_as_float(x.r[0]); im = __uint_as_float(x.r[1]);
  } else {
    re = x.re; im = x.im;
  }
}
template <typename R, bool TM> ME_DEV void xcset(R* sm, uint32_t tm, int off, R re, R im) {
  if constexpr (TM && sizeof(R) == 8) tm_st4(tm + ME_TM_COL(R, off), (uint32_t)__double2loint(re), (uint32_t)__double2hiint(re), (uint32_t)__double2loint(im), (uint32_t)__double2hiint(im));
  else if constexpr (TM) tm_st2(tm + ME_TM_COL(R, off), __float_as_uint(re), __float_as_uint(im));
  else cset<R>(sm + off, re, im);
}
// spinor basis (five reals) in an 8-slot TMEM vector
template <typename R, bool TM> ME_DEV SpinorBasis<R> xldsb(const R* sm, uint32_t tm, int off) {
  if constexpr (TM) {
    XW<R, TM> x; xldw_issue<R, TM>(x, sm, tm, off);
    const W4<R> w = xldw_get<R, TM>(x);
    SpinorBasis<R> g; g.a = w.r0; g.b = w.i0; g.c = w.r1; g.wp = w.i1; g.wm = w.r2; return g;
  } else {
    return ldsb<R>(sm + off);
  }
}
template <typename R, bool TM> ME_DEV void xstsb(R* sm, uint32_t tm, int off, const SpinorBasis<R>& g) {
  if constexpr (TM) xstw<R, TM>(sm, tm, off, W4<R>{g.a, g.b, g.c, g.wp, g.wm, (R)0, (R)0, (R)0});
  else stsb<R>(sm + off, g);
}
// ------------------------------------------------------------------------------------
// Current sharing across helicities (ME_OPT_SHARE_CURRENTS): a three-gluon sub-tree current depends on three gluon helicities
// only; the kernel parks it in a global scratch that stays resident in the 126 MB L2 (64 FP64 slots per thread do not fit on
// chip next to the rest) and reloads it on the steps of the helicity walk that leave those three helicities unchanged.
// Layout per CTA: [8-slot vector][4 pairs][ME_SM_STRIDE threads] of R2 (one coalesced 16-byte access per thread and pair, the
// vector index is an immediate offset); ld / st .cg: L2 only.
// ------------------------------------------------------------------------------------
template <typename R> ME_DEV void sc_stw(R* sc, int vec, const W4<R>& w) {
  typedef typename Pair2<R>::T R2;
  R2* q = reinterpret_cast<R2*>(sc) + vec * 4 * ME_SM_STRIDE;
  R2 a, b, c, d; a.x = w.r0; a.y = w.i0; b.x = w.r1; b.y = w.i1; c.x = w.r2; c.y = w.i2; d.x = w.r3; d.y = w.i3;
  __stcg(q, a); __stcg(q + ME_SM_STRIDE, b); __stcg(q + 2 * ME_SM_STRIDE, c); __stcg(q + 3 * ME_SM_STRIDE, d);
}
template <typename R> ME_DEV W4<R> sc_ldw(const R* sc, int vec) {
  typedef typename Pair2<R>::T R2;
  const R2* q = reinterpret_cast<const R2*>(sc) + vec * 4 * ME_SM_STRIDE;
  const R2 a = __ldcg(q), b = __ldcg(q + ME_SM_STRIDE), c = __ldcg(q + 2 * ME_SM_STRIDE), d = __ldcg(q + 3 * ME_SM_STRIDE);
  return {a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y};
}
// all earlier tcgen05.st of this thread are complete (needed before a tcgen05.ld that may read what they wrote)
template <bool TM> ME_DEV void xwait_st() {
  if constexpr (TM) asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
// TMEM allocation for one CTA of 128 threads: ncols columns (power of two >= 32), address of the warp's lane quarter returned
ME_DEV uint32_t tm_alloc(uint32_t* slot_in_smem, uint32_t ncols) {
  const int warp = threadIdx.x >> 5;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(slot_in_smem)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  return *slot_in_smem;
}
ME_DEV void tm_free(uint32_t base, uint32_t ncols) {
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if ((threadIdx.x >> 5) == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(ncols) : "memory");
}
}  // namespace me

#endif  // ME_HOST_FLOP_COUNT

// ------------------------------------------------------------------------------------
// Helpers of the orbit-looped kernels (codegen/emit_orbit.py): operands addressed through a
// per-instance table of shared-memory offsets, two-sided quark line, dual currents.
// ------------------------------------------------------------------------------------
namespace me {
template <typename R> ME_DEV Cx<R> cxs(const Cx<R>& c, R s) { return {c.re * s, c.im * s}; }
template <typename R> ME_DEV R lam_of(int h, int bit) { return ((h >> bit) & 1) ? (R)1 : (R)-1; }
// polarisation from a basis whose b part is pre-signed (+ for outgoing eps*, - for incoming eps)
template <typename R> ME_DEV W4<R> gluon_pol_from(const GluonBasis<R>& g, R lam) {
  return {(R)0, (R)0, -lam * g.ax, g.bx, -lam * g.ay, g.by, -lam * g.az, (R)0};
}
#ifndef ME_HOST_FLOP_COUNT
template <typename R> ME_DEV W4<R> gluon_pol_s(const R* p, R lam) { return gluon_pol_from<R>(ldgb<R>(p), lam); }
#endif
// column current grown from the t~ end: chi' = (q-slash + m) X * iden  (X = V-slash chi already formed)
template <typename R> ME_DEV W4<R> col_step(const W4<R>& X, const P4<R>& q, R m, R iden) {
  const R A = (q.e - q.z) * iden, B = (q.e + q.z) * iden, qx = q.x * iden, qy = q.y * iden, ms = m * iden;
  W4<R> o;
  // (qslash X)_0 = A X2 - C X3 ; _1 = -D X2 + B X3 ; _2 = B X0 + C X1 ; _3 = D X0 + A X1 ; C = qx - i qy, D = qx + i qy
  o.r0 = A * X.r2 - qx * X.r3 - qy * X.i3 + ms * X.r0;
  o.i0 = A * X.i2 - qx * X.i3 + qy * X.r3 + ms * X.i0;
  o.r1 = B * X.r3 - qx * X.r2 + qy * X.i2 + ms * X.r1;
  o.i1 = B * X.i3 - qx * X.i2 - qy * X.r2 + ms * X.i1;
  o.r2 = B * X.r0 + qx * X.r1 + qy * X.i1 + ms * X.r2;
  o.i2 = B * X.i0 + qx * X.i1 - qy * X.r1 + ms * X.i2;
  o.r3 = A * X.r1 + qx * X.r0 - qy * X.i0 + ms * X.r3;
  o.i3 = A * X.i1 + qx * X.i0 + qy * X.r0 + ms * X.i3;
  return o;
}
// row current grown from the t end: r' = r (q-slash + m) * iden  (r = psibar V-slash already formed); same arithmetic order
// as col_step (scale q once, then 4 products per component)
template <typename R> ME_DEV W4<R> row_step(const W4<R>& r, const P4<R>& q, R m, R iden) {
  const R A = (q.e - q.z) * iden, B = (q.e + q.z) * iden, qx = q.x * iden, qy = q.y * iden, ms = m * iden;
  W4<R> o;
  o.r2 = r.r0 * A - r.r1 * qx + r.i1 * qy + ms * r.r2;
  o.i2 = r.i0 * A - r.r1 * qy - r.i1 * qx + ms * r.i2;
  o.r3 = r.r1 * B - r.r0 * qx - r.i0 * qy + ms * r.r3;
  o.i3 = r.i1 * B - r.i0 * qx + r.r0 * qy + ms * r.i3;
  o.r0 = r.r2 * B + r.r3 * qx - r.i3 * qy + ms * r.r0;
  o.i0 = r.i2 * B + r.r3 * qy + r.i3 * qx + ms * r.i0;
  o.r1 = r.r3 * A + r.r2 * qx + r.i2 * qy + ms * r.r1;
  o.i1 = r.i3 * A + r.i2 * qx - r.r2 * qy + ms * r.i1;
  return o;
}
template <typename R> ME_DEV W4<R> quark_step2(const W4<R>& psibar, const W4<R>& V, const P4<R>& q, R m, R iden) {
  return row_step(row_slash(psibar, V), q, m, iden);
}
template <typename R> ME_DEV W4<R> wadd(const W4<R>& a, const W4<R>& b) {
  return {a.r0 + b.r0, a.i0 + b.i0, a.r1 + b.r1, a.i1 + b.i1, a.r2 + b.r2, a.i2 + b.i2, a.r3 + b.r3, a.i3 + b.i3};
}
template <typename R> ME_DEV W4<R> wsub(const W4<R>& a, const W4<R>& b) {
  return {a.r0 - b.r0, a.i0 - b.i0, a.r1 - b.r1, a.i1 - b.i1, a.r2 - b.r2, a.i2 - b.i2, a.r3 - b.r3, a.i3 - b.i3};
}
// dual of the three-gluon vertex:  v3_current(W1, W2, k1, k2, ik2) . J  ==  W1 . v3_dual(W2, J, k1, k2, ik2)
//   D = [ W2 ((k1-k2).J) + (k1+2k2) (W2.J) - J ((2k1+k2).W2) ] * ik2
template <typename R> ME_DEV W4<R> v3_dual(const W4<R>& W2, const W4<R>& J, const P4<R>& k1, const P4<R>& k2, R ik2) {
  const P4<R> d = psub(k1, k2);
  const P4<R> ka = {(k1.e + (R)2 * k2.e) * ik2, (k1.x + (R)2 * k2.x) * ik2, (k1.y + (R)2 * k2.y) * ik2, (k1.z + (R)2 * k2.z) * ik2};
  const P4<R> kb = {(R)2 * k1.e + k2.e, (R)2 * k1.x + k2.x, (R)2 * k1.y + k2.y, (R)2 * k1.z + k2.z};
  Cx<R> c1 = kdot(d, J), c3 = kdot(kb, W2);
  const Cx<R> c2 = wdot(W2, J);
  c1.re *= ik2; c1.im *= ik2; c3.re *= ik2; c3.im *= ik2;
  W4<R> o;
  o.r0 = c1.re * W2.r0 - c1.im * W2.i0 + c2.re * ka.e - c3.re * J.r0 + c3.im * J.i0;
  o.i0 = c1.re * W2.i0 + c1.im * W2.r0 + c2.im * ka.e - c3.re * J.i0 - c3.im * J.r0;
  o.r1 = c1.re * W2.r1 - c1.im * W2.i1 + c2.re * ka.x - c3.re * J.r1 + c3.im * J.i1;
  o.i1 = c1.re * W2.i1 + c1.im * W2.r1 + c2.im * ka.x - c3.re * J.i1 - c3.im * J.r1;
  o.r2 = c1.re * W2.r2 - c1.im * W2.i2 + c2.re * ka.y - c3.re * J.r2 + c3.im * J.i2;
  o.i2 = c1.re * W2.i2 + c1.im * W2.r2 + c2.im * ka.y - c3.re * J.i2 - c3.im * J.r2;
  o.r3 = c1.re * W2.r3 - c1.im * W2.i3 + c2.re * ka.z - c3.re * J.r3 + c3.im * J.i3;
  o.i3 = c1.re * W2.i3 + c1.im * W2.r3 + c2.im * ka.z - c3.re * J.i3 - c3.im * J.r3;
  return o;
}
}  // namespace me
