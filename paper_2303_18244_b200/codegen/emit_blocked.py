"""Blocked emitter for the single-kernel processes: register-pressure control by explicit storage classes.

The straight-line emitter of emit.py leaves every current to ptxas, which for g g -> t t~ g g spills
~40 KB per helicity to local memory and runs at <10 % of the FP64 pipe.  Here the generator decides:

  * per-event constants (momenta, 1/K^2, 1/(q^2-m^2), polarisation and spinor bases) and PERSISTENT
    currents (gluon sub-trees of 2..n-2 gluons, quark-line currents with 1..n-3 gluons attached) and
    the jamps live in per-thread shared-memory slots (BASELINE.json north_star: "jamp staging in
    shared memory"), layout [slot][thread] -> conflict-free, static offsets;
  * every other current is TRANSIENT: it has at most one transient operand, so the transient terms form
    a forest that is walked depth-first; each tree is one C++ scope whose values stay in registers and
    die at the closing brace.  Each diagram amplitude is consumed where it is produced.

Flop counting as in emit.py (routines of hel_amp.cuh as written).
"""
from .emit import FLOPS, bits, particle_of, colour_sum_lines, algorithmic_flops
from .topology import Topology


class BlockedEmitter:
    def __init__(self, T: Topology):
        self.T = T
        n = T.n
        self.n = n
        self.lines = []
        self.flops = 0
        self.namp = 0
        self.indent = 2
        # ---- storage classes
        self.persist_g = [g.id for g in T.G if 2 <= g.size <= n - 2]
        self.persist_q = [q.id for q in T.Q if 1 <= q.size <= n - 3]
        # ---- shared-memory slot map (units of R per thread)
        s = 0
        self.slot_mom = s; s += 4 * (n + 2)
        self.masks_k2 = [m for m in range(1, T.full + 1) if bin(m).count("1") >= 2]
        self.slot_ik2 = {m: s + i for i, m in enumerate(self.masks_k2)}; s += len(self.masks_k2)
        self.masks_q = [m for m in range(1, T.full)]
        self.slot_iq = {m: s + i for i, m in enumerate(self.masks_q)}; s += len(self.masks_q)
        self.slot_gb = {l: s + 5 * l for l in range(n)}; s += 5 * n
        self.slot_sbt = s; s += 5
        self.slot_sbtb = s; s += 5
        self.slot_g = {}
        for gid in self.persist_g:
            self.slot_g[gid] = s; s += 8
        self.slot_q = {}
        for qid in self.persist_q:
            self.slot_q[qid] = s; s += 8
        self.slot_j = s; s += 2 * T.ncol
        self.nslots = s
        # ---- consumer maps
        self.g_parents = {g.id: [] for g in T.G}
        for g in T.G:
            for c in set(g.ch):
                self.g_parents[c].append(g.id)
        self.q_of_g = {g.id: [] for g in T.G}     # quark terms attaching g
        self.q_children = {q.id: [] for q in T.Q}
        self.q_roots = []
        for q in T.Q:
            self.q_of_g[q.g].append(q.id)
            if q.prev >= 0:
                self.q_children[q.prev].append(q.id)
            else:
                self.q_roots.append(q.id)
        self.cl_of_g = {g.id: [] for g in T.G}
        self.cl_of_q = {q.id: [] for q in T.Q}
        self.cl_bare = []
        for c in T.Cl:
            self.cl_of_g[c.g].append(c.id)
            if c.q >= 0:
                self.cl_of_q[c.q].append(c.id)
            else:
                self.cl_bare.append(c.id)
        self.done_cl = set()
        self.scopes = []

    # ---------------------------------------------------------------- helpers
    def L(self, s):
        self.lines.append(" " * self.indent + s)

    def open(self):
        self.L("{")
        self.indent += 2
        self.scopes.append(set())

    def close(self):
        self.scopes.pop()
        self.indent -= 2
        self.L("}")

    def have(self, name):
        return any(name in s for s in self.scopes)

    def mark(self, name):
        self.scopes[-1].add(name)

    def is_persist_g(self, gid):
        return gid in self.slot_g

    def is_persist_q(self, qid):
        return qid in self.slot_q

    def is_transient_g(self, gid):
        return self.T.G[gid].size >= max(2, self.n - 1)

    def is_transient_q(self, qid):
        return self.T.Q[qid].size >= max(1, self.n - 2)

    def sgn(self, l):
        return 1 if l < 2 else -1

    def kvec(self, m):
        """make P4<R> K{m} (sum of incoming gluon momenta of the subset) available in the current scope"""
        name = "K%d" % m
        if self.have(name):
            return name
        comps = []
        b = bits(m)
        for ci in range(4):
            comps.append("".join(("+" if self.sgn(l) > 0 else "-") + "sm[%d * ME_SM_STRIDE]" % (self.slot_mom + 4 * particle_of(l) + ci) for l in b).lstrip("+"))
        self.L("const P4<R> %s = {%s};" % (name, ", ".join(comps)))
        self.flops += 4 * (len(b) - 1)
        self.mark(name)
        return name

    def qvec(self, m):
        """fermion-flow momentum p_t - K_m; for large subsets use K_complement - p_tbar"""
        name = "Q%d" % m
        if self.have(name):
            return name
        b = bits(m)
        comp = bits(self.T.full ^ m)
        comps = []
        if True:   # always p_t - K_S (no reliance on the input's momentum conservation)
            for ci in range(4):
                comps.append("sm[%d * ME_SM_STRIDE]" % (self.slot_mom + 8 + ci) +
                             "".join(("-" if self.sgn(l) > 0 else "+") + "sm[%d * ME_SM_STRIDE]" % (self.slot_mom + 4 * particle_of(l) + ci) for l in b))
            self.flops += 4 * len(b)
        else:
            for ci in range(4):
                comps.append("".join(("+" if self.sgn(l) > 0 else "-") + "sm[%d * ME_SM_STRIDE]" % (self.slot_mom + 4 * particle_of(l) + ci) for l in comp).lstrip("+") +
                             "-sm[%d * ME_SM_STRIDE]" % (self.slot_mom + 12 + ci))
            self.flops += 4 * len(comp)
        self.L("const P4<R> %s = {%s};" % (name, ", ".join(comps)))
        self.mark(name)
        return name

    def ik2(self, m):
        return "sm[%d * ME_SM_STRIDE]" % self.slot_ik2[m]

    def iq(self, m):
        return "sm[%d * ME_SM_STRIDE]" % self.slot_iq[m]

    def ref_g(self, gid):
        name = "g%d" % gid
        if self.have(name):
            return name
        g = self.T.G[gid]
        if g.kind == "leaf":
            lab = bits(g.mask)[0]
            self.L("const W4<R> %s = gluon_pol(ldgb<R>(sm, %d), lam%d, %s);" % (name, self.slot_gb[lab], particle_of(lab), "true" if lab >= 2 else "false"))
            self.flops += FLOPS["gluon_pol"]
        elif self.is_persist_g(gid):
            self.L("const W4<R> %s = ldw<R>(sm, %d);" % (name, self.slot_g[gid]))
        else:
            raise AssertionError("transient gluon term %d referenced out of scope" % gid)
        self.mark(name)
        return name

    def ref_q(self, qid):
        if qid < 0:
            return "ub"
        name = "q%d" % qid
        if self.have(name):
            return name
        assert self.is_persist_q(qid), "transient quark term %d referenced out of scope" % qid
        self.L("const W4<R> %s = ldw<R>(sm, %d);" % (name, self.slot_q[qid]))
        self.mark(name)
        return name

    def compute_g(self, gid):
        """emit the arithmetic of gluon term gid into the current scope (operands must be reachable)"""
        T = self.T
        g = T.G[gid]
        name = "g%d" % gid
        if g.kind == "v3":
            a, b = g.ch
            na, nb = self.ref_g(a), self.ref_g(b)
            ka, kb = self.kvec(T.G[a].mask), self.kvec(T.G[b].mask)
            self.L("const W4<R> %s = v3_current(%s, %s, %s, %s, %s);" % (name, na, nb, ka, kb, self.ik2(g.mask)))
            self.flops += FLOPS["v3_current"]
        else:
            a, b, c = g.ch
            k = int(g.kind[-1])
            na, nb, nc = self.ref_g(a), self.ref_g(b), self.ref_g(c)
            dn = "d%d_%d_%d" % (a, b, c)
            if not self.have(dn):
                self.L("const V4Dots<R> %s = v4_dots(%s, %s, %s, %s);" % (dn, na, nb, nc, self.ik2(g.mask)))
                self.flops += FLOPS["v4_dots"]
                self.mark(dn)
            self.L("const W4<R> %s = v4_current(%d, %s, %s, %s, %s);" % (name, k, dn, na, nb, nc))
            self.flops += FLOPS["v4_current"]
        self.mark(name)
        return name

    def compute_q(self, qid):
        q = self.T.Q[qid]
        name = "q%d" % qid
        prev = self.ref_q(q.prev)
        g = self.ref_g(q.g)
        qv = self.qvec(q.mask)
        self.L("const W4<R> %s = quark_step(%s, %s, %s, mt, %s);" % (name, prev, g, qv, self.iq(q.mask)))
        self.flops += FLOPS["quark_step"]
        self.mark(name)
        return name

    def jamp_update(self, cl, amp):
        for sigma, c in cl.jamp:
            jr = "sm[%d * ME_SM_STRIDE]" % (self.slot_j + 2 * sigma)
            ji = "sm[%d * ME_SM_STRIDE]" % (self.slot_j + 2 * sigma + 1)
            if c == 1:
                self.L("%s += %s.re; %s += %s.im;" % (jr, amp, ji, amp))
            elif c == -1:
                self.L("%s -= %s.re; %s -= %s.im;" % (jr, amp, ji, amp))
            elif c == 1j:
                self.L("%s -= %s.im; %s += %s.re;" % (jr, amp, ji, amp))
            elif c == -1j:
                self.L("%s += %s.im; %s -= %s.re;" % (jr, amp, ji, amp))
            else:
                raise AssertionError(c)
            self.flops += FLOPS["jamp_entry"]

    def closure(self, cid, vg_name=None):
        """amplitude of closure cid; its operands must be reachable.  vg_name: precomputed Vslash(g) v."""
        assert cid not in self.done_cl
        self.done_cl.add(cid)
        cl = self.T.Cl[cid]
        self.namp += 1
        if cl.q < 0:
            g = self.ref_g(cl.g)
            self.L("{ const Cx<R> a = wdot(%s, jtt);" % g)
            self.flops += FLOPS["wdot"]
        elif vg_name is not None:
            q = self.ref_q(cl.q)
            self.L("{ const Cx<R> a = row_col(%s, %s);" % (q, vg_name))
            self.flops += FLOPS["row_col"]
        else:
            q = self.ref_q(cl.q)
            g = self.ref_g(cl.g)
            self.L("{ const Cx<R> a = row_col(row_slash(%s, %s), vv);" % (q, g))
            self.flops += FLOPS["row_slash"] + FLOPS["row_col"]
        self.indent += 2
        self.jamp_update(cl, "a")
        self.indent -= 2
        self.L("}")

    # ---------------------------------------------------------------- the transient forest
    def node_g(self, gid):
        """transient gluon term: compute, then everything that consumes it"""
        self.open()
        name = self.compute_g(gid)
        # closures on the quark line with this g: share Vslash v
        cls = [c for c in self.cl_of_g[gid] if self.T.Cl[c].q >= 0]
        if cls:
            self.L("const W4<R> vg%d = slash_col(%s, vv);" % (gid, name))
            self.flops += FLOPS["slash_col"]
            for c in cls:
                self.closure(c, "vg%d" % gid)
        for c in self.cl_of_g[gid]:
            if self.T.Cl[c].q < 0:
                self.closure(c)
        for q in self.q_of_g[gid]:
            self.node_q(q)
        for p in self.g_parents[gid]:
            self.node_g(p)
        self.close()

    def node_q(self, qid):
        self.open()
        self.compute_q(qid)
        for c in self.cl_of_q[qid]:
            self.closure(c)
        for ch in self.q_children[qid]:
            self.node_q(ch)
        self.close()

    def transient_parent_count_g(self, gid):
        return sum(1 for c in set(self.T.G[gid].ch) if self.is_transient_g(c))

    def emit_helicity_body(self):
        T, n = self.T, self.n
        self.scopes = [set()]
        # phase A: persistent terms, in dependency order, each in its own scope
        for gid in self.persist_g:
            self.open()
            name = self.compute_g(gid)
            self.L("stw<R>(sm, %d, %s);" % (self.slot_g[gid], name))
            self.close()
        for qid in self.persist_q:
            self.open()
            name = self.compute_q(qid)
            self.L("stw<R>(sm, %d, %s);" % (self.slot_q[qid], name))
            self.close()
        # phase B: the transient forest
        for g in T.G:
            if self.is_transient_g(g.id) and self.transient_parent_count_g(g.id) == 0:
                self.node_g(g.id)
        for q in T.Q:
            if self.is_transient_q(q.id) and not (q.prev >= 0 and self.is_transient_q(q.prev)) and not self.is_transient_g(q.g):
                self.node_q(q.id)
        # closures whose operands are all persistent / leaves
        for c in T.Cl:
            if c.id not in self.done_cl:
                assert not self.is_transient_g(c.g) and (c.q < 0 or not self.is_transient_q(c.q)), c.id
                self.open()
                self.closure(c.id)
                self.close()
        assert len(self.done_cl) == len(T.Cl)

    # ---------------------------------------------------------------- per-event prologue
    def prologue(self):
        T, n = self.T, self.n
        P = []
        A = P.append
        fixed = 0
        sgn = self.sgn
        for i in range(n):
            for j in range(i + 1, n):
                A("const double d%d_%d = pdot(pd%d, pd%d);" % (i, j, particle_of(i), particle_of(j)))
                fixed += 7
        for l in range(n):
            A("const double dt%d = pdot(pd2, pd%d);" % (l, particle_of(l)))
            fixed += 7

        def k2expr(m):
            b = bits(m)
            terms = []
            for i in range(len(b)):
                for j in range(i + 1, len(b)):
                    s = sgn(b[i]) * sgn(b[j])
                    terms.append(("+" if s > 0 else "-") + "d%d_%d" % (b[i], b[j]))
            return "2.0*(" + "".join(terms).lstrip("+") + ")"

        for k in range(n + 2):
            A("stp<R>(sm, %d, pcast<R>(pd%d));" % (self.slot_mom + 4 * k, k))
        for m in self.masks_k2:
            A("sm[%d * ME_SM_STRIDE] = (R)(1.0/(%s));" % (self.slot_ik2[m], k2expr(m)))
            fixed += 2 + len(bits(m)) * (len(bits(m)) - 1) // 2
        for m in self.masks_q:
            b = bits(m)
            lin = "".join(("+" if sgn(l) > 0 else "-") + "dt%d" % l for l in b).lstrip("+")
            if len(b) == 1:
                A("sm[%d * ME_SM_STRIDE] = (R)(1.0/(-2.0*(%s)));" % (self.slot_iq[m], lin))
            else:
                A("sm[%d * ME_SM_STRIDE] = (R)(1.0/(%s-2.0*(%s)));" % (self.slot_iq[m], k2expr(m), lin))
            fixed += 4 + len(b) * (len(b) + 1) // 2
        for l in range(n):
            A("stgb<R>(sm, %d, gluon_basis(pcast<R>(pd%d)));" % (self.slot_gb[l], particle_of(l)))
            fixed += 20
        A("stsb<R>(sm, %d, spinor_basis(pcast<R>(pd2), mt));" % self.slot_sbt)
        A("stsb<R>(sm, %d, spinor_basis(pcast<R>(pd3), mt));" % self.slot_sbtb)
        fixed += 40
        self.fixed_flops = fixed
        return ["  " + s for s in P]


def emit_blocked_process(n, name, block=128):
    assert n >= 4, 'blocked emitter needs n >= 4 (forest property)'
    T = Topology(n)
    B = BlockedEmitter(T)
    B.indent = 4
    B.emit_helicity_body()
    pro = B.prologue()
    npar = n + 2
    ncol = T.ncol
    cs_lines, cs_flops = colour_sum_lines(T.color_num, ncol, T.color_denom)
    src = []
    S = src.append
    S("// GENERATED by paper_2303_18244_b200/codegen (blocked emitter) — do not edit.")
    S("// g g -> t t~ + %d g: %d diagrams, %d amplitudes, %d colour flows; %d shared-memory slots per thread." % (n - 2, T.ndiagrams, B.namp, ncol, B.nslots))
    S("#define ME_SM_STRIDE %d" % block)
    S("#include \"hel_amp.cuh\"")
    S("#include \"kernels.h\"")
    S("namespace me {")
    S("template <typename R, typename RC>")
    S("__global__ void __launch_bounds__(%d) k_%s(const double* __restrict__ mom, long n, long npad, const unsigned char* __restrict__ hels, int nhel,"
      " double mt_d, double norm_hel, double inv_avg, double* __restrict__ me_out, double* __restrict__ me_hel, double* __restrict__ jamp_out) {" % (block, name))
    S("  extern __shared__ __align__(16) unsigned char smem_raw[];")
    S("  R* sm = reinterpret_cast<R*>(smem_raw) + threadIdx.x;")
    S("  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;")
    S("  if (e >= npad) return;")
    S("  const R mt = (R)mt_d;")
    S("  {")
    S("  const double* pm = mom + (e >> 5) * (%d * 4 * 32) + (e & 31);" % npar)
    for k in range(npar):
        S("  const P4<double> pd%d = {pm[%d], pm[%d], pm[%d], pm[%d]};" % (k, (4 * k) * 32, (4 * k + 1) * 32, (4 * k + 2) * 32, (4 * k + 3) * 32))
    src.extend(pro)
    S("  }")
    S("  double acc = 0;")
    S("  for (int ih = 0; ih < nhel; ++ih) {")
    S("    const int h = hels[ih];")
    for k in range(npar):
        S("    const R lam%d = ((h >> %d) & 1) ? (R)1 : (R)-1;" % (k, npar - 1 - k))
    S("    const W4<R> ub = spinor_ubar(ldsb<R>(sm, %d), lam2);" % B.slot_sbt)
    S("    const W4<R> vv = spinor_v(ldsb<R>(sm, %d), lam3);" % B.slot_sbtb)
    S("    const W4<R> jtt = bilinear(ub, vv);")
    S("#pragma unroll")
    S("    for (int s = 0; s < %d; ++s) sm[(%d + s) * ME_SM_STRIDE] = 0;" % (2 * ncol, B.slot_j))
    src.extend(B.lines)
    S("    if (jamp_out != nullptr && e < n) {")
    S("#pragma unroll")
    S("      for (int s = 0; s < %d; ++s) jamp_out[(long)s * n + e] = (double)sm[(%d + s) * ME_SM_STRIDE];" % (2 * ncol, B.slot_j))
    S("    }")
    S("    RC cr[%d], ci[%d];" % (ncol, ncol))
    S("#pragma unroll")
    S("    for (int s = 0; s < %d; ++s) { cr[s] = (RC)sm[(%d + 2 * s) * ME_SM_STRIDE]; ci[s] = (RC)sm[(%d + 2 * s + 1) * ME_SM_STRIDE]; }" % (ncol, B.slot_j, B.slot_j))
    for l in cs_lines:
        S("    " + l)
    S("    const double meh = (double)cs;")
    S("    if (me_hel != nullptr && e < n) me_hel[(long)h * n + e] = meh * norm_hel;")
    S("    acc += meh;")
    S("  }")
    S("  if (me_out != nullptr && e < n) me_out[e] = acc * norm_hel * inv_avg;")
    S("}")
    per_hel = B.flops + cs_flops + 2 * FLOPS["spinor"] + FLOPS["bilinear"]
    S("static cudaError_t launch_%s(int precision, const LaunchArgs& a) {" % name)
    S("  const unsigned grid = (unsigned)((a.npad + %d - 1) / %d);" % (block, block))
    S("  const size_t smd = sizeof(double) * %d * %d, smf = sizeof(float) * %d * %d;" % (B.nslots, block, B.nslots, block))
    S("#define ME_ARGS a.mom, a.n, a.npad, a.hels, a.nhel, a.mt, a.norm_hel, a.inv_avg, a.me_out, a.me_hel, a.jamp_out")
    S("  if (precision == 0) {")
    S("    cudaFuncSetAttribute(k_%s<double, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smd);" % name)
    S("    k_%s<double, double><<<grid, %d, smd, a.stream>>>(ME_ARGS);" % (name, block))
    S("  } else if (precision == 1) {")
    S("    cudaFuncSetAttribute(k_%s<double, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smd);" % name)
    S("    k_%s<double, float><<<grid, %d, smd, a.stream>>>(ME_ARGS);" % (name, block))
    S("  } else {")
    S("    cudaFuncSetAttribute(k_%s<float, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smf);" % name)
    S("    k_%s<float, float><<<grid, %d, smf, a.stream>>>(ME_ARGS);" % (name, block))
    S("  }")
    S("#undef ME_ARGS")
    S("  return cudaGetLastError();")
    S("}")
    S("static const double color_num_%s[%d] = {%s};" % (name, ncol * ncol, ", ".join(str(float(x)) for row in T.color_num for x in row)))
    algo = algorithmic_flops(T)
    S("extern const ProcTable tab_%s = {%d, %d, %d, %d, %d, 1, {%r, %r, %r}, {%r, %r, %r}, %r, color_num_%s, launch_%s, nullptr};"
      % (name, n, T.ndiagrams, B.namp, ncol, T.color_denom, float(algo), float(algo), float(algo),
         float(per_hel), float(per_hel), float(per_hel), float(B.fixed_flops), name, name))
    S("}  // namespace me")
    info = dict(n=n, ndiagrams=T.ndiagrams, namp=B.namp, ncol=ncol, color_denom=T.color_denom, flops_per_helicity=algo,
                flops_executed_per_helicity=per_hel,
                fixed_flops=B.fixed_flops, colour_flops=cs_flops, smem_slots=B.nslots, block=block,
                persistent_g=len(B.persist_g), persistent_q=len(B.persist_q), color_num=T.color_num)
    return "\n".join(src) + "\n", info
