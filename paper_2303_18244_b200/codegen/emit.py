"""CUDA emitter: turns a Topology into straight-line per-helicity device code (one event per thread).

Emitted structure, per kernel:
  prologue  : load the event's momenta (AoSoA), build helicity-independent invariants in FP64
              (1/K^2 of every gluon subset, 1/(q^2-m^2) of every quark propagator, from pairwise
              dot products), gluon polarisation bases and spinor bases
  per helicity: external wavefunctions -> gluon sub-tree currents (by subset size) -> quark-line
              currents (by subset size) -> one amplitude per closure -> jamp accumulation
  flush     : colour sum J^dagger C J in-register, helicity accumulate.
Used for g g -> t t~ and g g -> t t~ g (everything fits the register file); the larger processes use the
orbit-looped emitters emit_orbit.py / emit_orbit5.py, which import the flop table and the colour-sum emitter from here.

Flop counting rule: add = mul = div = sqrt = 1, fma = 2, counted on the routines
of csrc/hel_amp.cuh as written.
"""
from .topology import Topology

# real flops of the routines in hel_amp.cuh, as written.  Not free parameters: tests/flopcount/count_flops.cpp instantiates the
# routines on the host with an operator-counting scalar and tests/test_abi_and_host.py compares every entry with what it counts
# (gluon_pol: the multiplication by the compile-time sign +-1 of eps / eps* is folded; spinor: either helicity branch).
FLOPS = dict(row_slash=64, slash_col=64, row_col=30, wdot=30, kdot=14, quark_step=127, v3_current=156,
             v4_dots=96, v4_current=56, bilinear=72, gluon_pol=3, spinor=6, jamp_entry=2)


def particle_of(label):
    return label if label < 2 else label + 2


# --- propagator denominators in double-double arithmetic (csrc/hel_amp.cuh "Propagator denominators")
DD_DOT_FLOPS = 4 * 2 + 3 * 17      # four error-free products, three double-double additions
DD_ADD_FLOPS = 17


def dd_sum(terms):
    """terms = [(sign, expression of type DD)] -> (nested dd_add / dd_sub expression, flops)"""
    sign, expr = terms[0]
    out = expr if sign > 0 else "dd_neg(%s)" % expr
    for sign, expr in terms[1:]:
        out = "%s(%s, %s)" % ("dd_add" if sign > 0 else "dd_sub", out, expr)
    return out, DD_ADD_FLOPS * (len(terms) - 1)


def dd_invariant_lines(labels, tlabels, sgn, part):
    """declarations of the exact pairwise invariants: d{i}_{j} = p_i.p_j, dt{l} = p_t.p_l, sq{l} = p_l^2, sqt = p_t^2 - m_t^2
    (labels: gluon labels that occur in a propagator; tlabels: those that occur in a quark propagator) -> (lines, flops)"""
    out, fl = [], 0
    labels = sorted(labels)
    for a, i in enumerate(labels):
        out.append("const DD sq%d = dd_dot(pd%d, pd%d);" % (i, part(i), part(i))); fl += DD_DOT_FLOPS
        for j in labels[a + 1:]:
            out.append("const DD d%d_%d = dd_dot(pd%d, pd%d);" % (i, j, part(i), part(j))); fl += DD_DOT_FLOPS
    if tlabels:
        out.append("const DD sqt = dd_offshell(pd2, mt_d);"); fl += DD_DOT_FLOPS + 2 + DD_ADD_FLOPS
    for l in sorted(tlabels):
        out.append("const DD dt%d = dd_dot(pd2, pd%d);" % (l, part(l))); fl += DD_DOT_FLOPS
    return out, fl


def dd_k2(b, sgn):
    """K^2 of the gluon set b (labels), K = sum_l sgn(l) p_l: sum_l p_l^2 + 2 sum_{i<j} sgn_i sgn_j p_i.p_j -> (DD expression, flops)"""
    terms = [(+1, "sq%d" % l) for l in b]
    pairs = [(sgn(b[i]) * sgn(b[j]), "d%d_%d" % (b[i], b[j])) for i in range(len(b)) for j in range(i + 1, len(b))]
    if pairs:
        pe, pf = dd_sum(pairs)
        terms.append((+1, "dd_mul2(%s)" % pe))
    else:
        pf = 0
    e, f = dd_sum(terms)
    return e, f + pf


def dd_q2(b, sgn):
    """(p_t - K)^2 - m_t^2 = (p_t^2 - m_t^2) + K^2 - 2 sum_l sgn(l) p_t.p_l -> (DD expression, flops)"""
    ke, kf = dd_k2(b, sgn)
    le, lf = dd_sum([(sgn(l), "dt%d" % l) for l in b])
    e, f = dd_sum([(+1, "sqt"), (+1, ke), (-1, "dd_mul2(%s)" % le)])
    return e, f + kf + lf


def bits(m):
    return [i for i in range(m.bit_length()) if m >> i & 1]


class KernelEmitter:
    """Emits the body of ONE kernel that evaluates a list of segments.
    segment = (closure ids, {colour index -> local jamp slot})."""

    def __init__(self, T: Topology):
        self.T = T
        self.lines = []          # per-helicity code
        self.done_g, self.done_q, self.done_vg, self.done_dots = set(), set(), set(), set()
        self.used_K, self.used_iK2, self.used_iQ, self.used_q = set(), set(), set(), set()
        self.flops = 0           # per helicity
        self.namp = 0
        self.have_jtt = False

    def L(self, s):
        self.lines.append("      " + s)

    # ---- gluon terms
    def need_g(self, gid):
        if gid in self.done_g:
            return
        T = self.T
        g = T.G[gid]
        if g.kind == "leaf":
            lab = bits(g.mask)[0]
            self.L("const W4<R> g%d = gluon_pol(gb%d, lam%d, %s);" % (gid, lab, particle_of(lab), "true" if lab >= 2 else "false"))
            self.flops += FLOPS["gluon_pol"]
        elif g.kind == "v3":
            a, b = g.ch
            self.need_g(a); self.need_g(b)
            ma, mb = T.G[a].mask, T.G[b].mask
            self.used_K.update((ma, mb)); self.used_iK2.add(g.mask)
            self.L("const W4<R> g%d = v3_current(g%d, g%d, K%d, K%d, iK2_%d);" % (gid, a, b, ma, mb, g.mask))
            self.flops += FLOPS["v3_current"]
        else:
            a, b, c = g.ch
            k = int(g.kind[-1])
            self.need_g(a); self.need_g(b); self.need_g(c)
            key = (a, b, c)
            if key not in self.done_dots:
                self.done_dots.add(key)
                self.used_iK2.add(g.mask)
                self.L("const V4Dots<R> d%d_%d_%d = v4_dots(g%d, g%d, g%d, iK2_%d);" % (a, b, c, a, b, c, g.mask))
                self.flops += FLOPS["v4_dots"]
            self.L("const W4<R> g%d = v4_current(%d, d%d_%d_%d, g%d, g%d, g%d);" % (gid, k, a, b, c, a, b, c))
            self.flops += FLOPS["v4_current"]
        self.done_g.add(gid)

    def need_q(self, qid):
        if qid < 0 or qid in self.done_q:
            return
        q = self.T.Q[qid]
        self.need_q(q.prev)
        self.need_g(q.g)
        self.used_q.add(q.mask); self.used_iQ.add(q.mask)
        prev = "ub" if q.prev < 0 else "q%d" % q.prev
        self.L("const W4<R> q%d = quark_step(%s, g%d, Q%d, mt, iQ_%d);" % (qid, prev, q.g, q.mask, q.mask))
        self.flops += FLOPS["quark_step"]
        self.done_q.add(qid)

    def need_vg(self, gid):
        if gid in self.done_vg:
            return
        self.need_g(gid)
        self.L("const W4<R> vg%d = slash_col(g%d, vv);" % (gid, gid))
        self.flops += FLOPS["slash_col"]
        self.done_vg.add(gid)

    def jamp_update(self, cl, jmap, amp):
        for sigma, c in cl.jamp:
            s = jmap[sigma]
            if c == 1:
                self.L("JR(%d) += %s.re; JI(%d) += %s.im;" % (s, amp, s, amp))
            elif c == -1:
                self.L("JR(%d) -= %s.re; JI(%d) -= %s.im;" % (s, amp, s, amp))
            elif c == 1j:
                self.L("JR(%d) -= %s.im; JI(%d) += %s.re;" % (s, amp, s, amp))
            elif c == -1j:
                self.L("JR(%d) += %s.im; JI(%d) -= %s.re;" % (s, amp, s, amp))
            else:
                raise AssertionError(c)
            self.flops += FLOPS["jamp_entry"]

    def emit_segment(self, closure_ids, jmap):
        T = self.T
        cls = [T.Cl[i] for i in closure_ids]
        # closures on the bare line: amp = g . (ubar gamma v)
        bare = [c for c in cls if c.q < 0]
        if bare and not self.have_jtt:
            self.L("const W4<R> jtt = bilinear(ub, vv);")
            self.flops += FLOPS["bilinear"]
            self.have_jtt = True
        for c in bare:
            self.need_g(c.g)
            self.L("{ const Cx<R> a = wdot(g%d, jtt);" % c.g)
            self.flops += FLOPS["wdot"]
            self.jamp_update(c, jmap, "a")
            self.L("}")
            self.namp += 1
        # quark-line closures, blocked by the quark mask so that Vslash v is shared
        rest = [c for c in cls if c.q >= 0]
        rest.sort(key=lambda c: (T.Q[c.q].size, T.Q[c.q].mask, c.q, c.g))
        for c in rest:
            self.need_q(c.q)
            self.need_vg(c.g)
            self.L("{ const Cx<R> a = row_col(q%d, vg%d);" % (c.q, c.g))
            self.flops += FLOPS["row_col"]
            self.jamp_update(c, jmap, "a")
            self.L("}")
            self.namp += 1

    # ---- helicity-independent prologue (FP64 invariants, cast to R)
    def prologue(self):
        T, n = self.T, self.T.n
        full = T.full
        self.smem_names = []
        P = []
        A = P.append
        sgn = lambda l: 1 if l < 2 else -1
        # which K vectors are needed: for K vectors, quark momenta
        need_K = set(self.used_K) | set(self.used_q)
        labs_needed = set()
        for m in need_K | self.used_iK2 | self.used_iQ:
            labs_needed.update(bits(m))
        fixed = 0
        # exact invariants (double-double) of the gluons that occur in a propagator
        labs, tl = set(), set()
        for m in self.used_iK2 | self.used_iQ:
            labs.update(bits(m))
        for m in self.used_iQ:
            tl.update(bits(m))
        lines, fl = dd_invariant_lines(labs, tl, sgn, particle_of)
        for l in lines:
            A(l)
        fixed += fl
        for m in sorted(self.used_iK2):
            e, fl = dd_k2(bits(m), sgn)
            A("const R iK2_%d = (R)(1.0 / dd_value(%s));" % (m, e))
            fixed += fl + 2
        for m in sorted(self.used_iQ):
            e, fl = dd_q2(bits(m), sgn)
            A("const R iQ_%d = (R)(1.0 / dd_value(%s));" % (m, e))
            fixed += fl + 2
        for m in sorted(need_K):
            b = bits(m)
            comps = []
            for c in "exyz":
                comps.append("".join(("+" if sgn(l) > 0 else "-") + "pd%d.%s" % (particle_of(l), c) for l in b).lstrip("+"))
            A("const P4<double> Kd%d = {%s};" % (m, ", ".join(comps)))
            fixed += 4 * (len(b) - 1)
            if m in self.used_K:
                if n in SMEM_KQ:      # FP64: parked in shared memory, reloaded at every use (volatile: the compiler must not keep it in a register)
                    A("const P4<R> K%dr = pcast<R>(Kd%d);" % (m, m))
                    A("if constexpr (sizeof(R) == 8) stp<R>(sm + ME_EO(%d), K%dr);" % (4 * len(self.smem_names), m)); self.smem_names.append("K%d" % m)
                else:
                    A("const P4<R> K%d = pcast<R>(Kd%d);" % (m, m))
            if m in self.used_q:
                if n in SMEM_KQ:
                    A("const P4<R> Q%dr = pcast<R>(psub(pd2, Kd%d));" % (m, m))
                    A("if constexpr (sizeof(R) == 8) stp<R>(sm + ME_EO(%d), Q%dr);" % (4 * len(self.smem_names), m)); self.smem_names.append("Q%d" % m)
                else:
                    A("const P4<R> Q%d = pcast<R>(psub(pd2, Kd%d));" % (m, m))
                fixed += 4
        self.smem_bases = []
        base_slot = 4 * len(self.smem_names)
        for l in range(n):
            if n in SMEM_KQ:
                A("const GluonBasis<R> gb%dr = gluon_basis(pcast<R>(pd%d));" % (l, particle_of(l)))
                A("if constexpr (sizeof(R) == 8) stgb<R>(sm, %d, gb%dr);" % (base_slot + 6 * len(self.smem_bases), l)); self.smem_bases.append(("gb%d" % l, "GluonBasis"))
            else:
                A("const GluonBasis<R> gb%d = gluon_basis(pcast<R>(pd%d));" % (l, particle_of(l)))
            fixed += 20
        for nm, pd in (("sbt", "pd2"), ("sbtb", "pd3")):
            if n in SMEM_KQ:
                A("const SpinorBasis<R> %sr = spinor_basis(pcast<R>(%s), mt);" % (nm, pd))
                A("if constexpr (sizeof(R) == 8) stsb<R>(sm, %d, %sr);" % (base_slot + 6 * len(self.smem_bases), nm)); self.smem_bases.append((nm, "SpinorBasis"))
            else:
                A("const SpinorBasis<R> %s = spinor_basis(pcast<R>(%s), mt);" % (nm, pd))
        fixed += 40
        self.fixed_flops = fixed
        return ["    " + s for s in P]


def colour_sum_lines(C, ncol, denom):
    """Triangular J^dagger C J (C real symmetric): 2*sum_i Jx_i*(C_ii/2 Jx_i + sum_{j>i} C_ij Jx_j), x in {r,i}."""
    out = []
    flops = 0
    out.append("RC cs = 0;")
    for part in ("cr", "ci"):
        for i in range(ncol):
            terms = ["(RC)%s*%s[%d]" % (repr(C[i][i] / 2.0), part, i)]
            flops += 1
            for j in range(i + 1, ncol):
                terms.append("(RC)%s*%s[%d]" % (repr(float(C[i][j])), part, j))
                flops += 2
            out.append("cs += %s[%d]*(%s);" % (part, i, " + ".join(terms)))
            flops += 2
    return out, flops


SMEM_KQ = {3}      # gluon counts whose kernel parks the helicity-independent momenta K_m, Q_m in shared memory instead of registers


def emit_single_kernel_process(n, name):
    """g g -> t t~ + (n-2) g evaluated by ONE kernel (n = 2,3,4): jamps in registers/local, in-kernel colour sum."""
    T = Topology(n)
    K = KernelEmitter(T)
    jmap = {s: s for s in range(T.ncol)}
    K.emit_segment([c.id for c in T.Cl], jmap)
    pro = K.prologue()
    cs_lines, cs_flops = colour_sum_lines(T.color_num, T.ncol, T.color_denom)
    npar = n + 2
    src = []
    S = src.append
    S("// GENERATED by paper_2303_18244_b200/codegen — do not edit.  g g -> t t~ + %d g: %d diagrams, %d amplitudes," % (n - 2, T.ndiagrams, K.namp))
    S("// %d gluon terms, %d quark terms, %d colour flows." % (len(K.done_g), len(K.done_q), T.ncol))
    S("#include \"hel_amp.cuh\"")
    S("#include \"kernels.h\"")
    S("namespace me {")
    if K.smem_names:
        S("// a four-momentum parked in shared memory (paired layout of hel_amp.cuh), loaded where it is used and not kept")
        S("// (FP32: registers suffice, the value computed in the prologue is returned as it is)")
        S("template <typename R> ME_DEV P4<R> ldpv(const R* p, const P4<R>& in_registers);")
        S("template <> ME_DEV P4<double> ldpv<double>(const double* p, const P4<double>&) {")
        S("  const unsigned a = (unsigned)__cvta_generic_to_shared(p); P4<double> v;")
        S("  asm volatile(\"ld.volatile.shared.v2.f64 {%0, %1}, [%2];\" : \"=d\"(v.e), \"=d\"(v.x) : \"r\"(a));")
        S("  asm volatile(\"ld.volatile.shared.v2.f64 {%%0, %%1}, [%%2 + %d];\" : \"=d\"(v.y), \"=d\"(v.z) : \"r\"(a));" % (16 * 128))
        S("  return v;")
        S("}")
        S("template <> ME_DEV P4<float> ldpv<float>(const float*, const P4<float>& in_registers) { return in_registers; }")
        S("// the same for the five numbers of a polarisation / spinor basis (both structs are five reals in the order ld5 / st5 store them)")
        S("template <typename R, typename B> ME_DEV B ld5v(const R* p, const B& in_registers) {")
        S("  if constexpr (sizeof(R) == 8) {")
        S("    const unsigned a = (unsigned)__cvta_generic_to_shared(p); double v[5];")
        S("    asm volatile(\"ld.volatile.shared.v2.f64 {%0, %1}, [%2];\" : \"=d\"(v[0]), \"=d\"(v[1]) : \"r\"(a));")
        S("    asm volatile(\"ld.volatile.shared.v2.f64 {%%0, %%1}, [%%2 + %d];\" : \"=d\"(v[2]), \"=d\"(v[3]) : \"r\"(a));" % (16 * 128))
        S("    asm volatile(\"ld.volatile.shared.f64 %%0, [%%1 + %d];\" : \"=d\"(v[4]) : \"r\"(a));" % (4 * 8 * 128))
        S("    return B{(R)v[0], (R)v[1], (R)v[2], (R)v[3], (R)v[4]};")
        S("  } else return in_registers;")
        S("}")
    S("#define JR(s) Jr[s]")
    S("#define JI(s) Ji[s]")
    S("template <typename R, typename RC>")
    S("__global__ void __launch_bounds__(ME_BLOCK) k_%s(const double* __restrict__ mom, long n, long npad, const unsigned char* __restrict__ hels, int nhel,"
      " double mt_d, double norm_hel, double inv_avg, double* __restrict__ me_out, double* __restrict__ me_hel, double* __restrict__ jamp_out,"
      " const int* __restrict__ helpe) {" % name)
    S("  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;")
    S("  if (e >= npad) return;")
    if K.smem_names:
        S("  extern __shared__ __align__(16) unsigned char smem_raw[];")
        S("  R* sm = reinterpret_cast<R*>(smem_raw) + 2 * threadIdx.x;")
    S("  const double* pm = mom + (e >> 5) * (%d * 4 * 32) + (e & 31);" % npar)
    for k in range(npar):
        S("  const P4<double> pd%d = {pm[%d], pm[%d], pm[%d], pm[%d]};" % (k, (4 * k) * 32, (4 * k + 1) * 32, (4 * k + 2) * 32, (4 * k + 3) * 32))
    S("  const R mt = (R)mt_d;")
    src.extend(pro)
    if K.smem_names:
        S("  ME_FENCE;      // the stores above are complete before the volatile loads below (their asm statements name no memory operand)")
    for i, nm in enumerate(K.smem_names):
        S("#define %s ldpv<R>(sm + ME_EO(%d), %sr)" % (nm, 4 * i, nm))
    for i, (nm, ty) in enumerate(K.smem_bases):
        S("#define %s ld5v<R, %s<R> >(sm + ME_EO(%d), %sr)" % (nm, ty, 4 * len(K.smem_names) + 6 * i, nm))
    S("  double acc = 0;")
    S("  for (int ih = 0; ih < nhel; ++ih) {")
    S("    const int h = helpe != nullptr ? helpe[e < n ? e : n - 1] : hels[ih];")
    for k in range(npar):
        S("    const R lam%d = ((h >> %d) & 1) ? (R)1 : (R)-1;" % (k, npar - 1 - k))
    S("    const W4<R> ub = spinor_ubar(sbt, lam2);")
    S("    const W4<R> vv = spinor_v(sbtb, lam3);")
    S("    R Jr[%d], Ji[%d];" % (T.ncol, T.ncol))
    S("#pragma unroll")
    S("    for (int s = 0; s < %d; ++s) { Jr[s] = 0; Ji[s] = 0; }" % T.ncol)
    S("    {")
    src.extend(K.lines)
    S("    }")
    S("    if (jamp_out != nullptr && e < n) {")
    S("#pragma unroll")
    S("      for (int s = 0; s < %d; ++s) { jamp_out[(2 * s) * n + e] = (double)Jr[s]; jamp_out[(2 * s + 1) * n + e] = (double)Ji[s]; }" % T.ncol)
    S("    }")
    S("    RC cr[%d], ci[%d];" % (T.ncol, T.ncol))
    S("#pragma unroll")
    S("    for (int s = 0; s < %d; ++s) { cr[s] = (RC)Jr[s]; ci[s] = (RC)Ji[s]; }" % T.ncol)
    for l in cs_lines:
        S("    " + l)
    S("    const double meh = (double)cs;")
    S("    if (me_hel != nullptr && e < n) me_hel[(long)h * n + e] = meh * norm_hel;")
    S("    acc += meh;")
    S("  }")
    S("  if (me_out != nullptr && e < n) me_out[e] = acc * norm_hel * inv_avg;")
    for nm in K.smem_names + [b for b, _ in K.smem_bases]:
        S("#undef %s" % nm)
    S("}")
    per_hel = K.flops + cs_flops + 2 * FLOPS["spinor"]
    S("static cudaError_t launch_%s(int precision, const LaunchArgs& a) {" % name)
    S("  const unsigned grid = (unsigned)((a.npad + ME_BLOCK - 1) / ME_BLOCK);")
    S("#define ME_ARGS a.mom, a.n, a.npad, a.hels, a.nhel, a.mt, a.norm_hel, a.inv_avg, a.me_out, a.me_hel, a.jamp_out, a.hel_per_event")
    nsl = 4 * len(K.smem_names) + 6 * len(K.smem_bases)
    S("  const size_t smd = sizeof(double) * %d * ME_BLOCK, smf = 0;" % nsl)
    if nsl:
        for inst, sm_ in (("double, double", "smd"), ("double, float", "smd"), ("float, float", "smf")):
            S("  cudaFuncSetAttribute(k_%s<%s>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)%s);" % (name, inst, sm_))
    S("  if (precision == 0) k_%s<double, double><<<grid, ME_BLOCK, smd, a.stream>>>(ME_ARGS);" % name)
    S("  else if (precision == 1) k_%s<double, float><<<grid, ME_BLOCK, smd, a.stream>>>(ME_ARGS);" % name)
    S("  else k_%s<float, float><<<grid, ME_BLOCK, smf, a.stream>>>(ME_ARGS);" % name)
    S("#undef ME_ARGS")
    S("  return cudaGetLastError();")
    S("}")
    S("static const double color_num_%s[%d] = {%s};" % (name, T.ncol * T.ncol, ", ".join(str(float(x)) for row in T.color_num for x in row)))
    S("extern const ProcTable tab_%s = {%d, %d, %d, %d, %d, 1, {%r, %r, %r}, {%r, %r, %r}, %r, color_num_%s, launch_%s, nullptr, false, nullptr, 0.0, 0, 0.0};"
      % (name, n, T.ndiagrams, K.namp, T.ncol, T.color_denom, float(per_hel), float(per_hel), float(per_hel),
         float(per_hel), float(per_hel), float(per_hel), float(K.fixed_flops), name, name))
    S("}  // namespace me")
    info = dict(n=n, ndiagrams=T.ndiagrams, namp=K.namp, ncol=T.ncol, color_denom=T.color_denom,
                flops_per_helicity=per_hel, fixed_flops=K.fixed_flops, colour_flops=cs_flops,
                n_gterms=len(K.done_g), n_qterms=len(K.done_q), color_num=T.color_num)
    return "\n".join(src) + "\n", info

