// =====================================================================================
// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, scalar CPU implementation of the tree-level matrix element |M|^2 of
//   cfg1  e+ e- -> mu+ mu-      cfg2  g g -> t t~        cfg3  g g -> t t~ g
//   cfg4  g g -> t t~ g g       cfg5  g g -> t t~ g g g
// written from the textbook Feynman rules (PAPER.md is a status report with no
// formulas: "based on Feynman diagrams and helicity amplitudes", "color
// algebra"; the readings are SURVEY.md §8(c) C1-C5, Q1-Q16, restated in DESIGN.md).
//
// It shares NO code with the CUDA path (paper_2303_18244_b200/): own diagram
// enumeration at run time, colour algebra done on explicit Lie polynomials, colour
// matrix computed numerically from Gell-Mann matrices, literal factors of i and g_s at
// every vertex and propagator.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may call it.
//
// Definition computed:
//   ME(p) = (1/D) sum_h sum_{sigma,tau} conj(J_sigma(p,h)) C_{sigma tau} J_tau(p,h)
// with J the colour-flow decomposition of the sum of all Feynman diagrams.
// ALL helicities are summed here (Q11); the helicity mask is a separate output (Q7).
//
// Pins: tests/test_oracle_*.py (closed forms cfg1/cfg2, Ward identity, Bose, Lorentz,
// parity, brute-force explicit colour, colour-matrix values, diagram counts, Philox
// known answers, RAMBO volumes, long double vs double, SURVEY worked examples).
// =====================================================================================
#include <algorithm>
#include <array>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <map>
#include <mutex>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace orc {

// ------------------------------------------------------------------------------------
// Basic types.  V4<R>: four complex numbers — either the contravariant components
// (0,1,2,3) of a Lorentz vector or the four components of a Dirac spinor in the chiral
// basis (components 0,1 = left-handed block, 2,3 = right-handed block).   [C1, C2]
// ------------------------------------------------------------------------------------
template <class R> using Cx = std::complex<R>;
template <class R> struct V4 { Cx<R> c[4]; };
template <class R> struct P4 { R c[4]; };  // real four-momentum (E,px,py,pz)

template <class R> static inline Cx<R> mdot(const V4<R>& a, const V4<R>& b) {  // metric (+,-,-,-)
  return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3];
}
template <class R> static inline Cx<R> mdot(const P4<R>& a, const V4<R>& b) {
  return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3];
}
template <class R> static inline R mdot(const P4<R>& a, const P4<R>& b) {
  return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3];
}

// ------------------------------------------------------------------------------------
// External states (conventions of Peskin & Schroeder App. A, chiral basis:
// gamma^0 = [[0,1],[1,0]], gamma^i = [[0,s^i],[-s^i,0]]).
// ------------------------------------------------------------------------------------
// two-spinors chi_lambda(p): helicity eigenstates of sigma.p^
template <class R> static void chi(const P4<R>& p, R pabs, int lam, Cx<R> out[2]) {
  const R pz = p.c[3];
  // |p|+pz, written as pT^2/(|p|-pz) in the backward hemisphere: same number, no cancellation
  // (DESIGN reading R4; the sum form loses digits like eps*|p|/(|p|+pz) close to the -z axis)
  const R ppz = pz >= R(0) ? pabs + pz : (p.c[1] * p.c[1] + p.c[2] * p.c[2]) / (pabs - pz);
  if (ppz == R(0)) {  // p along -z (always the case for beam particle 2), Q8
    if (lam > 0) { out[0] = 0; out[1] = 1; } else { out[0] = -1; out[1] = 0; }
    return;
  }
  const R N = R(1) / std::sqrt(R(2) * pabs * ppz);
  if (lam > 0) { out[0] = N * ppz; out[1] = N * Cx<R>(p.c[1], p.c[2]); }
  else         { out[0] = N * Cx<R>(-p.c[1], p.c[2]); out[1] = N * ppz; }
}
// omega_+- = sqrt(E +- |p|); massless legs take the explicit m=0 branch (|p|=E, omega_-=0).
template <class R> static void omegas(const P4<R>& p, R m, R& pabs, R& wp, R& wm) {
  if (m == R(0)) { pabs = p.c[0]; wp = std::sqrt(R(2) * p.c[0]); wm = 0; }
  else {
    pabs = std::sqrt(p.c[1] * p.c[1] + p.c[2] * p.c[2] + p.c[3] * p.c[3]);
    wp = std::sqrt(p.c[0] + pabs);
    wm = m / wp;  // = sqrt(E-|p|) on shell; avoids the cancellation in E-|p| (DESIGN reading R3)
  }
}
// u(p,lam) = (omega_{-lam} chi_lam , omega_{lam} chi_lam)
template <class R> static V4<R> spinor_u(const P4<R>& p, R m, int lam) {
  R pabs, wp, wm; omegas(p, m, pabs, wp, wm);
  Cx<R> x[2]; chi(p, pabs, lam, x);
  const R wl = lam > 0 ? wp : wm, wml = lam > 0 ? wm : wp;
  V4<R> u; u.c[0] = wml * x[0]; u.c[1] = wml * x[1]; u.c[2] = wl * x[0]; u.c[3] = wl * x[1];
  return u;
}
// v(p,lam) = (-lam omega_{lam} chi_{-lam} , lam omega_{-lam} chi_{-lam}); lam = physical helicity
template <class R> static V4<R> spinor_v(const P4<R>& p, R m, int lam) {
  R pabs, wp, wm; omegas(p, m, pabs, wp, wm);
  Cx<R> x[2]; chi(p, pabs, -lam, x);
  const R wl = lam > 0 ? wp : wm, wml = lam > 0 ? wm : wp;
  const R s = R(lam);
  V4<R> v; v.c[0] = -s * wl * x[0]; v.c[1] = -s * wl * x[1]; v.c[2] = s * wml * x[0]; v.c[3] = s * wml * x[1];
  return v;
}
// psi-bar = psi^dagger gamma^0 (row vector): swaps the two chirality blocks
template <class R> static V4<R> bar(const V4<R>& s) {
  V4<R> b; b.c[0] = std::conj(s.c[2]); b.c[1] = std::conj(s.c[3]); b.c[2] = std::conj(s.c[0]); b.c[3] = std::conj(s.c[1]);
  return b;
}
// polarisation vector eps(p,lam) = (-lam e1 - i e2)/sqrt2 (massless vector, eps^0 = 0)
template <class R> static V4<R> polvec(const P4<R>& p, int lam) {
  const R px = p.c[1], py = p.c[2], pz = p.c[3];
  const R pt = std::sqrt(px * px + py * py);
  const R pabs = std::sqrt(px * px + py * py + pz * pz);
  R e1[4], e2[4];
  if (pt == R(0)) {  // on the beam axis (always the case for the incoming gluons), Q8
    e1[0] = 0; e1[1] = 1; e1[2] = 0; e1[3] = 0;
    e2[0] = 0; e2[1] = 0; e2[2] = (pz >= 0 ? R(1) : R(-1)); e2[3] = 0;
  } else {
    e1[0] = 0; e1[1] = px * pz / (pabs * pt); e1[2] = py * pz / (pabs * pt); e1[3] = -pt / pabs;
    e2[0] = 0; e2[1] = -py / pt; e2[2] = px / pt; e2[3] = 0;
  }
  const R r = R(1) / std::sqrt(R(2));
  V4<R> e;
  for (int i = 0; i < 4; ++i) e.c[i] = Cx<R>(-R(lam) * e1[i] * r, -e2[i] * r);
  return e;
}
template <class R> static V4<R> conjv(const V4<R>& a) {
  V4<R> b; for (int i = 0; i < 4; ++i) b.c[i] = std::conj(a.c[i]); return b;
}

// ------------------------------------------------------------------------------------
// Dirac algebra in the chiral basis.  V-slash = [[0, V.sigma],[V.sigmabar, 0]] with
// V.sigma = V0 - V.s, V.sigmabar = V0 + V.s (2x2 blocks).
// ------------------------------------------------------------------------------------
template <class R> struct Slash { Cx<R> s[2][2], sb[2][2]; };  // V.sigma, V.sigmabar
template <class R> static Slash<R> slash(const V4<R>& V) {
  const Cx<R> I(0, 1);
  Slash<R> S;
  S.s[0][0] = V.c[0] - V.c[3];  S.s[0][1] = -(V.c[1] - I * V.c[2]);
  S.s[1][0] = -(V.c[1] + I * V.c[2]);  S.s[1][1] = V.c[0] + V.c[3];
  S.sb[0][0] = V.c[0] + V.c[3]; S.sb[0][1] = V.c[1] - I * V.c[2];
  S.sb[1][0] = V.c[1] + I * V.c[2]; S.sb[1][1] = V.c[0] - V.c[3];
  return S;
}
// column spinor:  (V-slash psi)
template <class R> static V4<R> slash_psi(const V4<R>& V, const V4<R>& psi) {
  Slash<R> S = slash(V); V4<R> o;
  o.c[0] = S.s[0][0] * psi.c[2] + S.s[0][1] * psi.c[3];
  o.c[1] = S.s[1][0] * psi.c[2] + S.s[1][1] * psi.c[3];
  o.c[2] = S.sb[0][0] * psi.c[0] + S.sb[0][1] * psi.c[1];
  o.c[3] = S.sb[1][0] * psi.c[0] + S.sb[1][1] * psi.c[1];
  return o;
}
// row spinor:  (psibar V-slash)
template <class R> static V4<R> psibar_slash(const V4<R>& pb, const V4<R>& V) {
  Slash<R> S = slash(V); V4<R> o;
  o.c[2] = pb.c[0] * S.s[0][0] + pb.c[1] * S.s[1][0];
  o.c[3] = pb.c[0] * S.s[0][1] + pb.c[1] * S.s[1][1];
  o.c[0] = pb.c[2] * S.sb[0][0] + pb.c[3] * S.sb[1][0];
  o.c[1] = pb.c[2] * S.sb[0][1] + pb.c[3] * S.sb[1][1];
  return o;
}
template <class R> static Cx<R> row_col(const V4<R>& row, const V4<R>& col) {
  return row.c[0] * col.c[0] + row.c[1] * col.c[1] + row.c[2] * col.c[2] + row.c[3] * col.c[3];
}
template <class R> static V4<R> p4_to_v4(const P4<R>& p) {
  V4<R> v; for (int i = 0; i < 4; ++i) v.c[i] = p.c[i]; return v;
}
// fermion current psibar gamma^mu psi (contravariant index mu)
template <class R> static V4<R> fermion_current(const V4<R>& pb, const V4<R>& psi) {
  V4<R> J;
  for (int mu = 0; mu < 4; ++mu) {
    V4<R> e; for (int i = 0; i < 4; ++i) e.c[i] = 0;
    // gamma^mu = slash of the covariant unit vector: V_nu gamma^nu with V_nu = delta_nu^mu,
    // i.e. contravariant V^mu = g^{mu mu}
    e.c[mu] = (mu == 0) ? 1 : -1;
    J.c[mu] = row_col(pb, slash_psi(e, psi));
  }
  return J;
}

// ------------------------------------------------------------------------------------
// Colour.  A colour factor is a polynomial in fundamental generators:
// map  (sequence of gluon labels)  ->  complex coefficient, meaning
//   sum_seq coef * T^{a_seq[0]} T^{a_seq[1]} ...
// ------------------------------------------------------------------------------------
typedef std::map<std::vector<int>, std::complex<double>> Poly;
static Poly pmul(const Poly& a, const Poly& b) {
  Poly r;
  for (auto& x : a) for (auto& y : b) {
    std::vector<int> s = x.first; s.insert(s.end(), y.first.begin(), y.first.end());
    r[s] += x.second * y.second;
  }
  return r;
}
static Poly padd(const Poly& a, const Poly& b, std::complex<double> cb) {
  Poly r = a; for (auto& y : b) r[y.first] += cb * y.second; return r;
}
static Poly pscale(const Poly& a, std::complex<double> c) { Poly r; for (auto& x : a) r[x.first] = c * x.second; return r; }
static Poly pcomm(const Poly& a, const Poly& b) { return padd(pmul(a, b), pmul(b, a), -1.0); }
static void pclean(Poly& a) {
  for (auto it = a.begin(); it != a.end();) { if (std::abs(it->second) < 1e-12) it = a.erase(it); else ++it; }
}

// Gell-Mann matrices lambda^a, T^a = lambda^a/2
static void gellmann(std::complex<double> T[8][3][3]) {
  typedef std::complex<double> Z; const Z I(0, 1);
  std::memset((void*)T, 0, sizeof(Z) * 72);
  T[0][0][1] = 1; T[0][1][0] = 1;
  T[1][0][1] = -I; T[1][1][0] = I;
  T[2][0][0] = 1; T[2][1][1] = -1;
  T[3][0][2] = 1; T[3][2][0] = 1;
  T[4][0][2] = -I; T[4][2][0] = I;
  T[5][1][2] = 1; T[5][2][1] = 1;
  T[6][1][2] = -I; T[6][2][1] = I;
  const double s3 = 1.0 / std::sqrt(3.0);
  T[7][0][0] = s3; T[7][1][1] = s3; T[7][2][2] = -2.0 * s3;
  for (int a = 0; a < 8; ++a) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) T[a][i][j] *= 0.5;
}

// ------------------------------------------------------------------------------------
// Diagram enumeration for g g -> t t~ + (n-2) g.
// Gluon labels 0..n-1: 0,1 = incoming g1,g2 (particles 0,1); 2.. = outgoing (particles 4..).
// A "gluon term" is one gluon sub-tree together with ONE colour structure (a 4-gluon
// vertex yields three terms); a "quark term" is a partial quark line grown from the
// outgoing t; a "closure" attaches the last gluon sub-tree and the outgoing t~.
// ------------------------------------------------------------------------------------
struct GTerm { int mask; int kind; int ch[3]; Poly col; bool canon; };   // kind 0 leaf, 1 V3, 2,3,4 = V4 structures 1,2,3
struct QTerm { int mask; int prev; int g; Poly col; bool canon; };       // prev=-1: bare ubar(p_t)
struct Closure { int q; int g; std::vector<std::pair<int, std::complex<double>>> jamp; bool canon; };

struct Topology {
  int n = 0, ncol = 0;
  std::vector<GTerm> G; std::vector<std::vector<int>> Gby;   // by mask
  std::vector<QTerm> Q; std::vector<std::vector<int>> Qby;
  std::vector<Closure> Cl;
  int ndiagrams = 0;
  std::vector<std::vector<int>> perms;                        // colour basis: permutations, lexicographic
  std::vector<double> C;                                      // colour matrix, ncol x ncol (numeric, real)
};

static int perm_index(const Topology& T, const std::vector<int>& s) {
  auto it = std::lower_bound(T.perms.begin(), T.perms.end(), s);
  return int(it - T.perms.begin());
}

static void build_topology(int n, Topology& T) {
  T.n = n;
  const int full = (1 << n) - 1;
  const std::complex<double> I(0, 1);
  T.Gby.assign(1 << n, {});
  // --- gluon sub-trees, by increasing subset size
  std::vector<int> masks; for (int m = 1; m <= full; ++m) masks.push_back(m);
  std::sort(masks.begin(), masks.end(), [](int a, int b) {
    int pa = __builtin_popcount(a), pb = __builtin_popcount(b); return pa != pb ? pa < pb : a < b; });
  for (int m : masks) {
    if (__builtin_popcount(m) == 1) {
      GTerm g; g.mask = m; g.kind = 0; g.ch[0] = g.ch[1] = g.ch[2] = -1; g.canon = true;
      g.col[{__builtin_ctz(m)}] = 1.0;
      T.Gby[m].push_back((int)T.G.size()); T.G.push_back(g);
      continue;
    }
    const int low = m & -m;
    // three-gluon vertex: unordered split {A,B}, A contains the lowest label
    for (int A = m; A > 0; A = (A - 1) & m) {
      if (!(A & low) || A == m) continue;
      const int B = m ^ A;
      for (int a : T.Gby[A]) for (int b : T.Gby[B]) {
        GTerm g; g.mask = m; g.kind = 1; g.ch[0] = a; g.ch[1] = b; g.ch[2] = -1;
        g.canon = T.G[a].canon && T.G[b].canon;
        // f^{abc} X1^a X2^b T^c = -i [X1, X2]
        g.col = pscale(pcomm(T.G[a].col, T.G[b].col), -I); pclean(g.col);
        T.Gby[m].push_back((int)T.G.size()); T.G.push_back(g);
      }
    }
    // four-gluon vertex: unordered split {A,B,C}; A has the lowest label, B the lowest of the rest
    for (int A = m; A > 0; A = (A - 1) & m) {
      if (!(A & low) || A == m) continue;
      const int rest = m ^ A, lowr = rest & -rest;
      for (int B = rest; B > 0; B = (B - 1) & rest) {
        if (!(B & lowr) || B == rest) continue;
        const int Cc = rest ^ B;
        for (int a : T.Gby[A]) for (int b : T.Gby[B]) for (int c : T.Gby[Cc]) {
          const Poly X1 = T.G[a].col, X2 = T.G[b].col, X3 = T.G[c].col;  // copies: T.G grows below
          for (int k = 0; k < 3; ++k) {
            GTerm g; g.mask = m; g.kind = 2 + k; g.ch[0] = a; g.ch[1] = b; g.ch[2] = c;
            g.canon = (k == 0) && T.G[a].canon && T.G[b].canon && T.G[c].canon;
            // f^{abe}f^{cde} -> -[[X1,X2],X3];  f^{ace}f^{bde} -> -[[X1,X3],X2];  f^{ade}f^{bce} -> [X1,[X2,X3]]
            if (k == 0) g.col = pscale(pcomm(pcomm(X1, X2), X3), -1.0);
            if (k == 1) g.col = pscale(pcomm(pcomm(X1, X3), X2), -1.0);
            if (k == 2) g.col = pcomm(X1, pcomm(X2, X3));
            pclean(g.col);
            T.Gby[m].push_back((int)T.G.size()); T.G.push_back(g);
          }
        }
      }
    }
  }
  // --- quark line grown from the outgoing t
  T.Qby.assign(1 << n, {});
  { QTerm q; q.mask = 0; q.prev = -1; q.g = -1; q.col[{}] = 1.0; q.canon = true; T.Qby[0].push_back(0); T.Q.push_back(q); }
  for (int m : masks) {
    if (m == full) continue;
    for (int A = m; A > 0; A = (A - 1) & m) {
      const int S = m ^ A;
      for (int q : T.Qby[S]) for (int g : T.Gby[A]) {
        QTerm t; t.mask = m; t.prev = q; t.g = g; t.canon = T.Q[q].canon && T.G[g].canon;
        t.col = pmul(T.Q[q].col, T.G[g].col);
        T.Qby[m].push_back((int)T.Q.size()); T.Q.push_back(t);
      }
    }
  }
  // --- colour basis and closures
  std::vector<int> id(n); for (int i = 0; i < n; ++i) id[i] = i;
  do { T.perms.push_back(id); } while (std::next_permutation(id.begin(), id.end()));
  T.ncol = (int)T.perms.size();
  T.ndiagrams = 0;
  for (int S = 0; S < full; ++S) {
    const int A = full ^ S;
    for (int q : T.Qby[S]) for (int g : T.Gby[A]) {
      Closure c; c.q = q; c.g = g; c.canon = T.Q[q].canon && T.G[g].canon;
      Poly col = pmul(T.Q[q].col, T.G[g].col); pclean(col);
      for (auto& x : col) c.jamp.push_back({perm_index(T, x.first), x.second});
      if (c.canon) ++T.ndiagrams;
      T.Cl.push_back(c);
    }
  }
  // --- colour matrix C_{sigma tau} = sum_{a_1..a_n} Tr( T^sigma (T^tau)^dagger ), numerically.
  // Row sigma = identity is computed from explicit Gell-Mann matrices; the other rows follow by
  // relabelling the summed colour indices: C_{sigma tau} = C_{id, sigma^-1 o tau}.
  typedef std::complex<double> Z;
  Z Tm[8][3][3]; gellmann(Tm);
  std::vector<Z> row(T.ncol, 0.0);
  std::vector<int> a(n, 0);
  long ncfg = 1; for (int i = 0; i < n; ++i) ncfg *= 8;
  for (long cfg = 0; cfg < ncfg; ++cfg) {
    long t = cfg; for (int i = 0; i < n; ++i) { a[i] = int(t % 8); t /= 8; }
    auto string_matrix = [&](const std::vector<int>& perm, Z M[3][3]) {
      Z A[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
      for (int k = 0; k < n; ++k) {
        Z B[3][3];
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
          B[i][j] = 0; for (int l = 0; l < 3; ++l) B[i][j] += A[i][l] * Tm[a[perm[k]]][l][j];
        }
        std::memcpy((void*)A, (void*)B, sizeof(A));
      }
      std::memcpy((void*)M, (void*)A, sizeof(A));
    };
    Z M0[3][3]; string_matrix(T.perms[0], M0);
    for (int tau = 0; tau < T.ncol; ++tau) {
      Z M1[3][3]; string_matrix(T.perms[tau], M1);
      Z s = 0; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) s += M0[i][j] * std::conj(M1[i][j]);
      row[tau] += s;
    }
  }
  T.C.assign((size_t)T.ncol * T.ncol, 0.0);
  for (int s = 0; s < T.ncol; ++s) for (int t = 0; t < T.ncol; ++t) {
    // rel = sigma^-1 o tau : position-wise, rel[k] = sigma^-1(tau[k])
    std::vector<int> inv(n), rel(n);
    for (int k = 0; k < n; ++k) inv[T.perms[s][k]] = k;
    for (int k = 0; k < n; ++k) rel[k] = inv[T.perms[t][k]];
    T.C[(size_t)s * T.ncol + t] = row[perm_index(T, rel)].real();
  }
}

static Topology& topology(int n) {
  static Topology T[8]; static std::once_flag once[8];
  std::call_once(once[n], [n]() { build_topology(n, T[n]); });
  return T[n];
}

// ------------------------------------------------------------------------------------
// Standard-Model parameters (SURVEY §8(b) me_sm_params; Q4-Q6)
// ------------------------------------------------------------------------------------
struct Params { double mz, wz, aewm1, sw2, mt, wt, alpha_s; };
static const long double PI_L = 3.14159265358979323846264338327950288L;

// ------------------------------------------------------------------------------------
// QCD processes: jamps for one event and one helicity.
// p[particle][4], particle order g g t t~ g...; hel[particle] = +-1.
// ward_leg >= 0: replace that gluon's polarisation by its momentum (Ward-identity pin).
// ------------------------------------------------------------------------------------
template <class R>
static void qcd_jamps(const Topology& T, const Params& prm, const P4<R>* p, const int* hel, int ward_leg,
                      std::vector<Cx<R>>& J) {
  const int n = T.n, full = (1 << n) - 1;
  const Cx<R> I(0, 1);
  const R gs = std::sqrt(R(4) * R(PI_L) * R(prm.alpha_s));
  const R mt = R(prm.mt);
  auto particle_of = [](int gl) { return gl < 2 ? gl : gl + 2; };
  // all-incoming gluon momenta and their subset sums
  std::vector<P4<R>> K(1 << n);
  for (int m = 0; m <= full; ++m) {
    for (int i = 0; i < 4; ++i) K[m].c[i] = 0;
    for (int gl = 0; gl < n; ++gl) if (m >> gl & 1) {
      const R sgn = gl < 2 ? R(1) : R(-1);
      for (int i = 0; i < 4; ++i) K[m].c[i] += sgn * p[particle_of(gl)].c[i];
    }
  }
  // gluon sub-tree currents
  std::vector<V4<R>> Gc(T.G.size());
  for (size_t t = 0; t < T.G.size(); ++t) {
    const GTerm& g = T.G[t];
    if (g.kind == 0) {
      const int gl = __builtin_ctz(g.mask), ip = particle_of(gl);
      if (gl == ward_leg) Gc[t] = p4_to_v4(p[ip]);
      else { V4<R> e = polvec(p[ip], hel[ip]); Gc[t] = gl < 2 ? e : conjv(e); }  // incoming eps, outgoing eps*
      continue;
    }
    const P4<R>& Km = K[g.mask];
    const R K2 = mdot(Km, Km);
    const Cx<R> prop = -I / K2;                               // -i g^{mu nu} / k^2 (Feynman gauge)
    if (g.kind == 1) {
      const V4<R>&V1 = Gc[g.ch[0]], &V2 = Gc[g.ch[1]];
      const P4<R>&k1 = K[T.G[g.ch[0]].mask], &k2 = K[T.G[g.ch[1]].mask];
      P4<R> k3; for (int i = 0; i < 4; ++i) k3.c[i] = -Km.c[i];  // third leg, incoming convention
      // g_s [ g^{mu nu}(k1-k2)^rho + g^{nu rho}(k2-k3)^mu + g^{rho mu}(k3-k1)^nu ] V1_mu V2_nu
      P4<R> d12, d23, d31;
      for (int i = 0; i < 4; ++i) { d12.c[i] = k1.c[i] - k2.c[i]; d23.c[i] = k2.c[i] - k3.c[i]; d31.c[i] = k3.c[i] - k1.c[i]; }
      const Cx<R> v12 = mdot(V1, V2), a = mdot(d23, V1), b = mdot(d31, V2);
      for (int i = 0; i < 4; ++i) Gc[t].c[i] = prop * gs * (v12 * d12.c[i] + a * V2.c[i] + b * V1.c[i]);
    } else {
      const V4<R>&V1 = Gc[g.ch[0]], &V2 = Gc[g.ch[1]], &V3 = Gc[g.ch[2]];
      const Cx<R> v12 = mdot(V1, V2), v13 = mdot(V1, V3), v23 = mdot(V2, V3);
      const Cx<R> vf = -I * gs * gs;                          // -i g_s^2 [ ... ]
      for (int i = 0; i < 4; ++i) {
        Cx<R> kin;
        if (g.kind == 2) kin = v13 * V2.c[i] - v23 * V1.c[i];       // g^{mu rho}g^{nu sig} - g^{mu sig}g^{nu rho}
        else if (g.kind == 3) kin = v12 * V3.c[i] - v23 * V1.c[i];  // g^{mu nu}g^{rho sig} - g^{mu sig}g^{nu rho}
        else kin = v12 * V3.c[i] - v13 * V2.c[i];                   // g^{mu nu}g^{rho sig} - g^{mu rho}g^{nu sig}
        Gc[t].c[i] = prop * vf * kin;
      }
    }
  }
  // quark line from the outgoing t:  psibar_new = psibar_old (i g_s V-slash) i(q-slash + m)/(q^2 - m^2)
  const P4<R>& pt = p[2]; const P4<R>& ptb = p[3];
  std::vector<V4<R>> Qc(T.Q.size());
  for (size_t t = 0; t < T.Q.size(); ++t) {
    const QTerm& q = T.Q[t];
    if (q.prev < 0) { Qc[t] = bar(spinor_u(pt, mt, hel[2])); continue; }
    P4<R> qm; for (int i = 0; i < 4; ++i) qm.c[i] = pt.c[i] - K[q.mask].c[i];
    const R den = mdot(qm, qm) - mt * mt;
    V4<R> r = psibar_slash(Qc[q.prev], Gc[q.g]);
    for (int i = 0; i < 4; ++i) r.c[i] *= I * gs;
    V4<R> rq = psibar_slash(r, p4_to_v4(qm));
    for (int i = 0; i < 4; ++i) Qc[t].c[i] = I * (rq.c[i] + mt * r.c[i]) / den;
  }
  // closures on the outgoing t~
  const V4<R> v = spinor_v(ptb, mt, hel[3]);
  J.assign(T.ncol, Cx<R>(0));
  for (const Closure& c : T.Cl) {
    const Cx<R> amp = I * gs * row_col(Qc[c.q], slash_psi(Gc[c.g], v));
    for (auto& e : c.jamp) J[e.first] += Cx<R>(R(e.second.real()), R(e.second.imag())) * amp;
  }
}

template <class R>
static R colour_sum(const Topology& T, const std::vector<Cx<R>>& J) {
  Cx<R> s = 0;
  for (int a = 0; a < T.ncol; ++a) for (int b = 0; b < T.ncol; ++b)
    s += std::conj(J[a]) * R(T.C[(size_t)a * T.ncol + b]) * J[b];
  return s.real();
}

// cfg1: e+(p0) e-(p1) -> mu+(p2) mu-(p3), s-channel photon + Z
template <class R>
static R epem_me_hel(const Params& prm, const P4<R>* p, const int* hel) {
  const Cx<R> I(0, 1);
  const R e = std::sqrt(R(4) * R(PI_L) / R(prm.aewm1));
  const R sw2 = R(prm.sw2), sw = std::sqrt(sw2), cw = std::sqrt(R(1) - sw2);
  const R gL = (R(-0.5) + sw2) / (sw * cw), gR = sw2 / (sw * cw);
  const R mz = R(prm.mz), wz = R(prm.wz);
  P4<R> k; for (int i = 0; i < 4; ++i) k.c[i] = p[0].c[i] + p[1].c[i];
  const R s = mdot(k, k);
  // incoming antifermion e+: vbar(p0); incoming fermion e-: u(p1); outgoing mu-: ubar(p3); outgoing mu+: v(p2)
  const V4<R> vb = bar(spinor_v(p[0], R(0), hel[0])), u = spinor_u(p[1], R(0), hel[1]);
  const V4<R> ub = bar(spinor_u(p[3], R(0), hel[3])), v = spinor_v(p[2], R(0), hel[2]);
  auto PL = [](const V4<R>& x) { V4<R> y = x; y.c[2] = 0; y.c[3] = 0; return y; };  // gamma5 = diag(-1,-1,1,1)
  auto PR = [](const V4<R>& x) { V4<R> y = x; y.c[0] = 0; y.c[1] = 0; return y; };
  // photon: (-i e gamma^mu) (-i g_{mu nu}/s) (-i e gamma^nu)
  const V4<R> Je = fermion_current(vb, u), Jm = fermion_current(ub, v);
  Cx<R> amp = (-I * e) * (-I / s) * (-I * e) * mdot(Je, Jm);
  // Z: (i e gamma^mu (gL PL + gR PR)) (-i g_{mu nu}/(s - mz^2 + i mz wz)) (same vertex)
  V4<R> JeZ, JmZ;
  { V4<R> a = fermion_current(vb, PL(u)), b = fermion_current(vb, PR(u));
    for (int i = 0; i < 4; ++i) JeZ.c[i] = gL * a.c[i] + gR * b.c[i]; }
  { V4<R> a = fermion_current(ub, PL(v)), b = fermion_current(ub, PR(v));
    for (int i = 0; i < 4; ++i) JmZ.c[i] = gL * a.c[i] + gR * b.c[i]; }
  amp += (I * e) * (-I / (Cx<R>(s - mz * mz, mz * wz))) * (I * e) * mdot(JeZ, JmZ);
  return std::norm(amp);
}

struct ProcInfo { int npar, nglu, ncomb, avg_denom; };
static bool proc_info(int process, ProcInfo& pi) {
  switch (process) {
    case 0: pi = {4, 0, 16, 4}; return true;
    case 1: pi = {4, 2, 16, 256}; return true;
    case 2: pi = {5, 3, 32, 256}; return true;
    case 3: pi = {6, 4, 64, 512}; return true;      // 4*64*2!
    case 4: pi = {7, 5, 128, 1536}; return true;    // 4*64*3!
  }
  return false;
}

// per-helicity colour-summed |M_h|^2 (no averaging) for one event
template <class R>
static void me_event(int process, const Params& prm, const double* pd, int ward_leg, double* me_hel_out, double* me_out) {
  ProcInfo pi; proc_info(process, pi);
  P4<R> p[8];
  for (int k = 0; k < pi.npar; ++k) for (int i = 0; i < 4; ++i) p[k].c[i] = R(pd[4 * k + i]);
  R tot = 0;
  std::vector<Cx<R>> J;
  for (int ih = 0; ih < pi.ncomb; ++ih) {
    int hel[8];
    for (int k = 0; k < pi.npar; ++k) hel[k] = (ih >> (pi.npar - 1 - k) & 1) ? +1 : -1;   // C1: particle 1 = MSB
    R mh;
    if (process == 0) mh = epem_me_hel<R>(prm, p, hel);
    else { const Topology& T = topology(pi.nglu); qcd_jamps<R>(T, prm, p, hel, ward_leg, J); mh = colour_sum<R>(T, J); }
    if (me_hel_out) me_hel_out[ih] = double(mh);
    tot += mh;
  }
  *me_out = double(tot / R(pi.avg_denom));
}

// ------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11) and the uniform mapping of SURVEY Q14
// ------------------------------------------------------------------------------------
static void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c[4] = {ctr_in[0], ctr_in[1], ctr_in[2], ctr_in[3]}, k[2] = {key_in[0], key_in[1]};
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)M0 * c[0], p1 = (uint64_t)M1 * c[2];
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0, hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c[1] ^ k[0], n1 = lo1, n2 = hi0 ^ c[3] ^ k[1], n3 = lo0;
    c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
    k[0] += W0; k[1] += W1;
  }
  for (int i = 0; i < 4; ++i) out[i] = c[i];
}
static inline double u53(uint32_t a, uint32_t b) {   // ((a>>5)*2^26 + (b>>6) + 0.5) * 2^-53, in (0,1)
  return ((double)(a >> 5) * 67108864.0 + (double)(b >> 6) + 0.5) * (1.0 / 9007199254740992.0);
}

// ------------------------------------------------------------------------------------
// RAMBO (Kleiss, Stirling, Ellis 1986), SURVEY Q12.  Final state in the CM frame at sqrt_s.
// ------------------------------------------------------------------------------------
template <class R>
static void rambo_event(int nf, const double* mass, double sqrt_s_d, const double* rnd, double* pout, double* wt) {
  const R sqs = R(sqrt_s_d), PI = R(PI_L);
  R q[8][4], Q[4] = {0, 0, 0, 0};
  for (int k = 0; k < nf; ++k) {
    const R r1 = R(rnd[4 * k]), r2 = R(rnd[4 * k + 1]), r3 = R(rnd[4 * k + 2]), r4 = R(rnd[4 * k + 3]);
    const R c = R(2) * r1 - R(1), phi = R(2) * PI * r2, q0 = -std::log(r3 * r4), s = std::sqrt(R(1) - c * c);
    q[k][0] = q0; q[k][1] = q0 * s * std::cos(phi); q[k][2] = q0 * s * std::sin(phi); q[k][3] = q0 * c;
    for (int i = 0; i < 4; ++i) Q[i] += q[k][i];
  }
  const R M = std::sqrt(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
  const R b[3] = {-Q[1] / M, -Q[2] / M, -Q[3] / M}, x = sqs / M, gam = Q[0] / M, a = R(1) / (R(1) + gam);
  R pk[8][4];
  for (int k = 0; k < nf; ++k) {
    const R bq = b[0] * q[k][1] + b[1] * q[k][2] + b[2] * q[k][3];
    for (int i = 0; i < 3; ++i) pk[k][1 + i] = x * (q[k][1 + i] + b[i] * q[k][0] + a * bq * b[i]);
    // energy of the boosted massless momentum: x (gam q0 + b.q) == |p| algebraically.  The conformal boost amplifies rounding
    // by (Q0/M)^2 (up to ~1e8 among 5e5 events), which would leave the first form off shell by up to 4e-4 GeV^2; |p| keeps every
    // momentum on its mass shell to rounding (reading Q12a)
    pk[k][0] = std::sqrt(pk[k][1] * pk[k][1] + pk[k][2] * pk[k][2] + pk[k][3] * pk[k][3]);
    (void)gam;
  }
  // massless weight: (pi/2)^{n-1} s^{n-2} / ((n-1)!(n-2)!) * (2 pi)^{4-3n}
  R fact1 = 1, fact2 = 1; for (int i = 2; i <= nf - 1; ++i) fact1 *= i; for (int i = 2; i <= nf - 2; ++i) fact2 *= i;
  R w = std::pow(PI / R(2), nf - 1) * std::pow(sqs * sqs, nf - 2) / (fact1 * fact2) * std::pow(R(2) * PI, 4 - 3 * nf);
  bool massive = false; R summ = 0;
  for (int k = 0; k < nf; ++k) { if (mass[k] != 0.0) massive = true; summ += R(mass[k]); }
  if (massive) {
    R xi = std::sqrt(R(1) - (summ / sqs) * (summ / sqs));
    for (int it = 0; it < 100; ++it) {
      R f = -sqs, df = 0;
      for (int k = 0; k < nf; ++k) {
        const R e = std::sqrt(R(mass[k]) * R(mass[k]) + xi * xi * pk[k][0] * pk[k][0]);
        f += e; df += xi * pk[k][0] * pk[k][0] / e;
      }
      if (std::fabs(f) < R(1e-14) * sqs) break;
      xi -= f / df;
    }
    R prod = 1, sum2 = 0;
    for (int k = 0; k < nf; ++k) {
      const R e = std::sqrt(R(mass[k]) * R(mass[k]) + xi * xi * pk[k][0] * pk[k][0]);
      for (int i = 1; i < 4; ++i) pk[k][i] *= xi;
      pk[k][0] = e;
      const R k3 = std::sqrt(pk[k][1] * pk[k][1] + pk[k][2] * pk[k][2] + pk[k][3] * pk[k][3]);
      prod *= k3 / e; sum2 += k3 * k3 / e;
    }
    w *= std::pow(xi, 2 * nf - 3) * prod * sqs / sum2;
  }
  // beams along +-z, massless (C1)
  pout[0] = double(sqs / 2); pout[1] = 0; pout[2] = 0; pout[3] = double(sqs / 2);
  pout[4] = double(sqs / 2); pout[5] = 0; pout[6] = 0; pout[7] = double(-sqs / 2);
  for (int k = 0; k < nf; ++k) for (int i = 0; i < 4; ++i) pout[4 * (2 + k) + i] = double(pk[k][i]);
  if (wt) *wt = double(w);
}

}  // namespace orc

// =====================================================================================
// C interface for ctypes (tests, smoke, bench cpu_baseline).  Momenta are AoS
// [event][particle][4] doubles here; layout conversion lives in the input module.
// =====================================================================================
extern "C" {

int orc_info(int process, int* out /* npar, nglu, ncomb, avg_denom, ncol, ndiagrams, n_gterms, n_qterms, n_closures */) {
  orc::ProcInfo pi; if (!orc::proc_info(process, pi)) return 1;
  out[0] = pi.npar; out[1] = pi.nglu; out[2] = pi.ncomb; out[3] = pi.avg_denom;
  if (process == 0) { out[4] = 1; out[5] = 2; out[6] = out[7] = out[8] = 0; return 0; }
  const orc::Topology& T = orc::topology(pi.nglu);
  out[4] = T.ncol; out[5] = T.ndiagrams; out[6] = (int)T.G.size(); out[7] = (int)T.Q.size(); out[8] = (int)T.Cl.size();
  return 0;
}

// number of gluon sub-tree topologies G(k) for the full k-gluon set (4-vertex counted once), SURVEY C4
int orc_count_gluon_subtrees(int n) {
  const orc::Topology& T = orc::topology(n); int c = 0;
  for (int g : T.Gby[(1 << n) - 1]) if (T.G[g].canon) ++c;
  return c;
}

int orc_color_matrix(int process, double* out) {
  orc::ProcInfo pi; if (!orc::proc_info(process, pi) || process == 0) return 1;
  const orc::Topology& T = orc::topology(pi.nglu);
  std::memcpy(out, T.C.data(), sizeof(double) * T.C.size());
  return 0;
}

// params: mz, wz, aewm1, sw2, mt, wt, alpha_s
int orc_me(int process, const double* params, const double* p, long n, int use_long_double, int ward_leg,
           double* me, double* me_hel /* nullable, [n][ncomb] */, int nthreads) {
  orc::ProcInfo pi; if (!orc::proc_info(process, pi)) return 1;
  orc::Params prm; std::memcpy(&prm, params, sizeof(prm));
  if (process != 0) orc::topology(pi.nglu);  // build outside the parallel region
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 4) num_threads(nthreads)
#endif
  for (long e = 0; e < n; ++e) {
    const double* pe = p + (size_t)e * pi.npar * 4;
    double* mh = me_hel ? me_hel + (size_t)e * pi.ncomb : nullptr;
    if (use_long_double) orc::me_event<long double>(process, prm, pe, ward_leg, mh, me + e);
    else orc::me_event<double>(process, prm, pe, ward_leg, mh, me + e);
  }
  return 0;
}

// jamps of one event and one helicity index (QCD processes), out[ncol][2]
int orc_jamps(int process, const double* params, const double* p, int ihel, double* out) {
  orc::ProcInfo pi; if (!orc::proc_info(process, pi) || process == 0) return 1;
  orc::Params prm; std::memcpy(&prm, params, sizeof(prm));
  const orc::Topology& T = orc::topology(pi.nglu);
  orc::P4<double> pp[8]; int hel[8];
  for (int k = 0; k < pi.npar; ++k) { for (int i = 0; i < 4; ++i) pp[k].c[i] = p[4 * k + i]; hel[k] = (ihel >> (pi.npar - 1 - k) & 1) ? 1 : -1; }
  std::vector<orc::Cx<double>> J; orc::qcd_jamps<double>(T, prm, pp, hel, -1, J);
  for (int a = 0; a < T.ncol; ++a) { out[2 * a] = J[a].real(); out[2 * a + 1] = J[a].imag(); }
  return 0;
}

// Event-by-event helicity / leading-colour choice (rule stated in include/me.h
// me_select_helicity_color and DESIGN.md "Selection"): u1,u2 from Philox counter (event lo, event hi, 'SELE', 0);
// inverse CDF in index order over ME_h of the good helicities, then over |J_s|^2 at the chosen helicity.
static int orc_inverse_cdf(const std::vector<double>& w, double u) {
  double tot = 0; for (double x : w) tot += x;
  const double target = u * tot;
  double cum = 0; int sel = -1, lastpos = 0;
  for (size_t k = 0; k < w.size(); ++k) {
    cum += w[k];
    if (w[k] > 0) lastpos = (int)k;
    if (sel < 0 && w[k] > 0 && cum >= target) sel = (int)k;
  }
  return sel < 0 ? lastpos : sel;
}
int orc_select(int process, const double* params, const double* p, long n, uint64_t seed, uint64_t first_event,
               const uint64_t* mask, int* ihel, int* icol) {
  orc::ProcInfo pi; if (!orc::proc_info(process, pi)) return 1;
  orc::Params prm; std::memcpy(&prm, params, sizeof(prm));
  if (process != 0) orc::topology(pi.nglu);
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 4)
#endif
  for (long e = 0; e < n; ++e) {
    const double* pe = p + (size_t)e * pi.npar * 4;
    std::vector<double> mh(pi.ncomb); double tot;
    orc::me_event<double>(process, prm, pe, -1, mh.data(), &tot);
    for (int h = 0; h < pi.ncomb; ++h) if (!(mask[h >> 6] >> (h & 63) & 1)) mh[h] = 0;
    const uint64_t ev = first_event + (uint64_t)e;
    const uint32_t ctr[4] = {(uint32_t)ev, (uint32_t)(ev >> 32), 0x53454C45u, 0u};
    uint32_t w[4]; orc::philox4x32_10(ctr, key, w);
    const double u1 = orc::u53(w[0], w[1]), u2 = orc::u53(w[2], w[3]);
    ihel[e] = orc_inverse_cdf(mh, u1);
    if (process == 0) { icol[e] = 0; continue; }
    const orc::Topology& T = orc::topology(pi.nglu);
    orc::P4<double> pp[8]; int hel[8];
    for (int k = 0; k < pi.npar; ++k) { for (int i = 0; i < 4; ++i) pp[k].c[i] = pe[4 * k + i]; hel[k] = (ihel[e] >> (pi.npar - 1 - k) & 1) ? 1 : -1; }
    std::vector<orc::Cx<double>> J; orc::qcd_jamps<double>(T, prm, pp, hel, -1, J);
    std::vector<double> wj(T.ncol);
    for (int a = 0; a < T.ncol; ++a) wj[a] = std::norm(J[a]);
    icol[e] = orc_inverse_cdf(wj, u2);
  }
  return 0;
}

// first uniform of Philox counter (event lo, event hi, tag, 0), key = seed: the per-event random number of the
// unweighting step (tag 'UNWT', include/me.h me_unweight)
void orc_tagged_uniform(uint64_t seed, uint64_t first_event, long n, uint32_t tag, double* out) {
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  for (long e = 0; e < n; ++e) {
    const uint64_t ev = first_event + (uint64_t)e;
    const uint32_t ctr[4] = {(uint32_t)ev, (uint32_t)(ev >> 32), tag, 0u};
    uint32_t w[4]; orc::philox4x32_10(ctr, key, w);
    out[e] = orc::u53(w[0], w[1]);
  }
}

int orc_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// external-state primitives (for the invariants of SURVEY C2). kind: 0 u, 1 v, 2 eps. out[4][2]
void orc_external(int kind, const double* p, double m, int lam, double* out) {
  orc::P4<double> pp; for (int i = 0; i < 4; ++i) pp.c[i] = p[i];
  orc::V4<double> w = kind == 0 ? orc::spinor_u(pp, m, lam) : kind == 1 ? orc::spinor_v(pp, m, lam) : orc::polvec(pp, lam);
  for (int i = 0; i < 4; ++i) { out[2 * i] = w.c[i].real(); out[2 * i + 1] = w.c[i].imag(); }
}

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { orc::philox4x32_10(ctr, key, out); }

// out[n][per_event][4] uniforms in (0,1); SURVEY Q14
void orc_philox_uniform(uint64_t seed, uint64_t first_event, long n, int per_event, double* out) {
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  for (long e = 0; e < n; ++e) {
    const uint64_t ev = first_event + (uint64_t)e;
    for (int k = 0; k < per_event; ++k) {
      uint32_t w[8];
      for (int j = 0; j < 2; ++j) {
        const uint32_t ctr[4] = {(uint32_t)ev, (uint32_t)(ev >> 32), (uint32_t)k, (uint32_t)j};
        orc::philox4x32_10(ctr, key, w + 4 * j);
      }
      double* o = out + ((size_t)e * per_event + k) * 4;
      for (int i = 0; i < 4; ++i) o[i] = orc::u53(w[2 * i], w[2 * i + 1]);
    }
  }
}

// rnd[n][nfinal][4] -> p[n][2+nfinal][4], wt[n] (nullable)
int orc_rambo(int nfinal, const double* masses, double sqrt_s, const double* rnd, long n, double* p, double* wt, int use_long_double) {
  if (nfinal < 2 || nfinal > 6) return 1;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
  for (long e = 0; e < n; ++e) {
    const double* r = rnd + (size_t)e * nfinal * 4;
    double* po = p + (size_t)e * (2 + nfinal) * 4;
    if (use_long_double) orc::rambo_event<long double>(nfinal, masses, sqrt_s, r, po, wt ? wt + e : nullptr);
    else orc::rambo_event<double>(nfinal, masses, sqrt_s, r, po, wt ? wt + e : nullptr);
  }
  return 0;
}

}  // extern "C"
