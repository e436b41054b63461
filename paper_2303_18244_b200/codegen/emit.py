"""CUDA emitter: turns a Topology into straight-line per-helicity device code (one event per thread).

Emitted structure, per kernel:
  prologue  : load the event's momenta (AoSoA), build helicity-independent invariants in FP64
              (1/K^2 of every gluon subset, 1/(q^2-m^2) of every quark propagator, from pairwise
              dot products), gluon polarisation bases and spinor bases
  per helicity: external wavefunctions -> gluon sub-tree currents (by subset size) -> quark-line
              currents (by subset size) -> one amplitude per closure -> jamp accumulation
  flush     : single-kernel processes: colour sum J^dagger C J in-register, helicity accumulate;
              multi-kernel process (g g -> t t~ g g g): add the segment's jamps into the global
              staging buffer consumed by the batched colour-sum kernel.

Flop counting rule: add = mul = div = sqrt = 1, fma = 2, counted on the routines
of csrc/hel_amp.cuh as written.
"""
from .topology import Topology

# real flops of the routines in hel_amp.cuh, as written
FLOPS = dict(row_slash=64, slash_col=64, row_col=30, wdot=30, kdot=14, quark_step=131, v3_current=156,
             v4_dots=96, v4_current=56, bilinear=72, gluon_pol=3, spinor=8, jamp_entry=2)


def particle_of(label):
    return label if label < 2 else label + 2


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
        P = []
        A = P.append
        sgn = lambda l: 1 if l < 2 else -1
        # which K vectors are needed: for K vectors, quark momenta
        need_K = set(self.used_K) | set(self.used_q)
        labs_needed = set()
        for m in need_K | self.used_iK2 | self.used_iQ:
            labs_needed.update(bits(m))
        fixed = 0
        # pairwise invariants
        pairs = set()
        for m in self.used_iK2 | self.used_iQ:
            b = bits(m)
            for i in range(len(b)):
                for j in range(i + 1, len(b)):
                    pairs.add((b[i], b[j]))
        for (i, j) in sorted(pairs):
            A("const double d%d_%d = pdot(pd%d, pd%d);" % (i, j, particle_of(i), particle_of(j)))
            fixed += 7
        tl = set()
        for m in self.used_iQ:
            tl.update(bits(m))
        for l in sorted(tl):
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

        for m in sorted(self.used_iK2):
            A("const R iK2_%d = (R)(1.0/(%s));" % (m, k2expr(m)))
            fixed += 2 + len(bits(m)) * (len(bits(m)) - 1) // 2
        for m in sorted(self.used_iQ):
            b = bits(m)
            lin = "".join(("+" if sgn(l) > 0 else "-") + "dt%d" % l for l in b).lstrip("+")
            if len(b) == 1:
                A("const R iQ_%d = (R)(1.0/(-2.0*(%s)));" % (m, lin))
            else:
                A("const R iQ_%d = (R)(1.0/(%s-2.0*(%s)));" % (m, k2expr(m), lin))
            fixed += 4 + len(b) * (len(b) + 1) // 2
        for m in sorted(need_K):
            b = bits(m)
            comps = []
            for c in "exyz":
                comps.append("".join(("+" if sgn(l) > 0 else "-") + "pd%d.%s" % (particle_of(l), c) for l in b).lstrip("+"))
            A("const P4<double> Kd%d = {%s};" % (m, ", ".join(comps)))
            fixed += 4 * (len(b) - 1)
            if m in self.used_K:
                A("const P4<R> K%d = pcast<R>(Kd%d);" % (m, m))
            if m in self.used_q:
                A("const P4<R> Q%d = pcast<R>(psub(pd2, Kd%d));" % (m, m))
                fixed += 4
        for l in range(n):
            A("const GluonBasis<R> gb%d = gluon_basis(pcast<R>(pd%d));" % (l, particle_of(l)))
            fixed += 20
        A("const SpinorBasis<R> sbt = spinor_basis(pcast<R>(pd2), mt);")
        A("const SpinorBasis<R> sbtb = spinor_basis(pcast<R>(pd3), mt);")
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


def algorithmic_flops(T):
    """Single-pass count: every gluon term, quark term, Vslash.v product and amplitude exactly once, jamp adds,
    triangular colour sum (ncol <= 24) or dense contraction (ncol = 120), external spinors."""
    K = KernelEmitter(T)
    K.emit_segment([c.id for c in T.Cl], {s: s for s in range(T.ncol)})
    if T.ncol <= 24:
        cs = colour_sum_lines(T.color_num, T.ncol, T.color_denom)[1]
    else:
        cs = 2 * (2 * T.ncol * T.ncol) + 4 * T.ncol
    return K.flops + cs + 2 * FLOPS["spinor"]


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
    S("#define JR(s) Jr[s]")
    S("#define JI(s) Ji[s]")
    S("template <typename R, typename RC>")
    S("__global__ void __launch_bounds__(ME_BLOCK) k_%s(const double* __restrict__ mom, long n, long npad, const unsigned char* __restrict__ hels, int nhel,"
      " double mt_d, double norm_hel, double inv_avg, double* __restrict__ me_out, double* __restrict__ me_hel, double* __restrict__ jamp_out,"
      " const int* __restrict__ helpe) {" % name)
    S("  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;")
    S("  if (e >= npad) return;")
    S("  const double* pm = mom + (e >> 5) * (%d * 4 * 32) + (e & 31);" % npar)
    for k in range(npar):
        S("  const P4<double> pd%d = {pm[%d], pm[%d], pm[%d], pm[%d]};" % (k, (4 * k) * 32, (4 * k + 1) * 32, (4 * k + 2) * 32, (4 * k + 3) * 32))
    S("  const R mt = (R)mt_d;")
    src.extend(pro)
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
    S("}")
    per_hel = K.flops + cs_flops + 2 * FLOPS["spinor"]
    S("static cudaError_t launch_%s(int precision, const LaunchArgs& a) {" % name)
    S("  const unsigned grid = (unsigned)((a.npad + ME_BLOCK - 1) / ME_BLOCK);")
    S("#define ME_ARGS a.mom, a.n, a.npad, a.hels, a.nhel, a.mt, a.norm_hel, a.inv_avg, a.me_out, a.me_hel, a.jamp_out, a.hel_per_event")
    S("  if (precision == 0) k_%s<double, double><<<grid, ME_BLOCK, 0, a.stream>>>(ME_ARGS);" % name)
    S("  else if (precision == 1) k_%s<double, float><<<grid, ME_BLOCK, 0, a.stream>>>(ME_ARGS);" % name)
    S("  else k_%s<float, float><<<grid, ME_BLOCK, 0, a.stream>>>(ME_ARGS);" % name)
    S("#undef ME_ARGS")
    S("  return cudaGetLastError();")
    S("}")
    S("static const double color_num_%s[%d] = {%s};" % (name, T.ncol * T.ncol, ", ".join(str(float(x)) for row in T.color_num for x in row)))
    S("extern const ProcTable tab_%s = {%d, %d, %d, %d, %d, 1, {%r, %r, %r}, {%r, %r, %r}, %r, color_num_%s, launch_%s, nullptr};"
      % (name, n, T.ndiagrams, K.namp, T.ncol, T.color_denom, float(per_hel), float(per_hel), float(per_hel),
         float(per_hel), float(per_hel), float(per_hel), float(K.fixed_flops), name, name))
    S("}  // namespace me")
    info = dict(n=n, ndiagrams=T.ndiagrams, namp=K.namp, ncol=T.ncol, color_denom=T.color_denom,
                flops_per_helicity=per_hel, fixed_flops=K.fixed_flops, colour_flops=cs_flops,
                n_gterms=len(K.done_g), n_qterms=len(K.done_q), color_num=T.color_num)
    return "\n".join(src) + "\n", info


# ==========================================================================================
# g g -> t t~ g g g: diagrams split across kernels (BASELINE.json north_star: "Register-pressure
# control for the 1240-diagram case comes from splitting the diagrams across kernels"), jamps
# staged in global memory and summed by the batched colour kernel (csrc/color_sum.cu).
# ==========================================================================================
JMAX = 48            # local jamp accumulators per segment (shared memory, [2*JMAX][ME_BLOCK])
KERNEL_CLOSURES = 60


def _chain_key(T, c):
    """Gluon-subset masks along the quark line from the t end; bare-line closures are keyed by the top-level split."""
    if c.q < 0:
        g = T.G[c.g]
        return (tuple(sorted(T.G[x].mask for x in g.ch)), (g.mask,))
    ms = [T.G[c.g].mask]
    q = c.q
    while q >= 0:
        ms.append(T.G[T.Q[q].g].mask)
        q = T.Q[q].prev
    return ((), tuple(reversed(ms)))


def partition(T, jmax=None, kernel_closures=None):
    """-> list of kernels, each a list of segments (closure ids, sorted support)."""
    jmax = jmax or JMAX
    kernel_closures = kernel_closures or KERNEL_CLOSURES
    cl = sorted(T.Cl, key=lambda c: (_chain_key(T, c), c.q, c.g))
    segs, cur, sup = [], [], set()
    for c in cl:
        s = set(j for j, _ in c.jamp)
        if cur and (len(sup | s) > jmax or len(cur) >= kernel_closures):
            segs.append((cur, sorted(sup))); cur, sup = [], set()
        cur.append(c.id); sup |= s
    segs.append((cur, sorted(sup)))
    kernels, curk, cnt = [], [], 0
    for sg in segs:
        if curk and cnt + len(sg[0]) > kernel_closures:
            kernels.append(curk); curk, cnt = [], 0
        curk.append(sg); cnt += len(sg[0])
    kernels.append(curk)
    return kernels


def emit_multi_kernel_process(n, name):
    T = Topology(n)
    kernels = partition(T)
    npar = n + 2
    files = {}
    touched = set()
    total_flops, total_namp, fixed_max = 0, 0, 0
    kinfo = []
    for ki, segs in enumerate(kernels):
        K = KernelEmitter(T)
        body = []
        for (cids, sup) in segs:
            jmap = {sigma: slot for slot, sigma in enumerate(sup)}
            K.lines = []
            K.emit_segment(cids, jmap)
            body.extend(K.lines)
            # flush this segment's jamps into the global staging buffer, then clear the slots
            for sigma in sup:
                op = "+=" if sigma in touched else "="
                touched.add(sigma)
                body.append("      gj[%dL * npad] %s (RJ)JR(%d); gj[%dL * npad] %s (RJ)JI(%d); JR(%d) = 0; JI(%d) = 0;"
                            % (2 * sigma, op, jmap[sigma], 2 * sigma + 1, op, jmap[sigma], jmap[sigma], jmap[sigma]))
                if op == "+=":
                    K.flops += 2
        pro = K.prologue()
        src = []
        S = src.append
        S("// GENERATED by paper_2303_18244_b200/codegen — do not edit.  g g -> t t~ g g g, diagram kernel %d of %d:" % (ki, len(kernels)))
        S("// %d amplitudes in %d segments; %d gluon terms, %d quark terms evaluated here." % (K.namp, len(segs), len(K.done_g), len(K.done_q)))
        S("#include \"hel_amp.cuh\"")
        S("#include \"kernels.h\"")
        S("#include \"multi.h\"")
        S("namespace me {")
        S("#define JR(s) sj[(2 * (s)) * ME_BLOCK]")
        S("#define JI(s) sj[(2 * (s) + 1) * ME_BLOCK]")
        S("template <typename R, typename RJ>")
        S("__global__ void __launch_bounds__(ME_BLOCK) k_%s_p%d(const double* __restrict__ mom, long npad, const unsigned char* __restrict__ hels,"
          " double mt_d, RJ* __restrict__ gjbase) {" % (name, ki))
        S("  extern __shared__ __align__(16) unsigned char smem_raw[];")
        S("  R* sj = reinterpret_cast<R*>(smem_raw) + threadIdx.x;")
        S("  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;")
        S("  if (e >= npad) return;")
        S("  const double* pm = mom + (e >> 5) * (%d * 4 * 32) + (e & 31);" % npar)
        for k in range(npar):
            S("  const P4<double> pd%d = {pm[%d], pm[%d], pm[%d], pm[%d]};" % (k, (4 * k) * 32, (4 * k + 1) * 32, (4 * k + 2) * 32, (4 * k + 3) * 32))
        S("  const R mt = (R)mt_d;")
        src.extend(pro)
        S("  {")
        S("    const int h = hels[blockIdx.y];")
        S("    RJ* gj = gjbase + (long)blockIdx.y * (%d * 2) * npad + e;" % T.ncol)
        for k in range(npar):
            S("    const R lam%d = ((h >> %d) & 1) ? (R)1 : (R)-1;" % (k, npar - 1 - k))
        S("    const W4<R> ub = spinor_ubar(sbt, lam2);")
        S("    const W4<R> vv = spinor_v(sbtb, lam3);")
        S("#pragma unroll")
        S("    for (int s = 0; s < %d; ++s) { JR(s) = 0; JI(s) = 0; }" % JMAX)
        S("    {")
        src.extend(body)
        S("    }")
        S("  }")
        S("}")
        S("static cudaError_t launch_p%d(int precision, const MultiArgs& a) {" % ki)
        S("  const dim3 grid((unsigned)((a.npad + ME_BLOCK - 1) / ME_BLOCK), (unsigned)a.nh);")
        S("  if (precision == 2) {")
        S("    const size_t sm = sizeof(float) * 2 * %d * ME_BLOCK;" % JMAX)
        S("    cudaFuncSetAttribute(k_%s_p%d<float, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);" % (name, ki))
        S("    k_%s_p%d<float, float><<<grid, ME_BLOCK, sm, a.stream>>>(a.mom, a.npad, a.hels, a.mt, (float*)a.gj);" % (name, ki))
        S("  } else {")
        S("    const size_t sm = sizeof(double) * 2 * %d * ME_BLOCK;" % JMAX)
        S("    cudaFuncSetAttribute(k_%s_p%d<double, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);" % (name, ki))
        S("    k_%s_p%d<double, double><<<grid, ME_BLOCK, sm, a.stream>>>(a.mom, a.npad, a.hels, a.mt, (double*)a.gj);" % (name, ki))
        S("  }")
        S("  return cudaGetLastError();")
        S("}")
        S("extern const MultiKernel mk_%s_p%d = {launch_p%d};" % (name, ki, ki))
        S("}  // namespace me")
        files["gen_%s_p%d.cu" % (name, ki)] = "\n".join(src) + "\n"
        total_flops += K.flops + 2 * FLOPS["spinor"]
        total_namp += K.namp
        fixed_max += K.fixed_flops
        kinfo.append(dict(amplitudes=K.namp, segments=len(segs), gterms=len(K.done_g), qterms=len(K.done_q), flops=K.flops))
    assert touched == set(range(T.ncol))
    # colour sum as a dense contraction: 2 * ncol * (2 ncol) FMA-flops + 4 ncol for the final dot
    cs_flops = 2 * (2 * T.ncol * T.ncol) + 4 * T.ncol
    per_hel = total_flops + cs_flops
    src = []
    S = src.append
    S("// GENERATED by paper_2303_18244_b200/codegen — do not edit.  g g -> t t~ g g g process table.")
    S("#include \"kernels.h\"")
    S("#include \"multi.h\"")
    S("namespace me {")
    for ki in range(len(kernels)):
        S("extern const MultiKernel mk_%s_p%d;" % (name, ki))
    S("static const MultiKernel* const parts_%s[%d] = {%s};" % (name, len(kernels), ", ".join("&mk_%s_p%d" % (name, ki) for ki in range(len(kernels)))))
    S("static const double color_num_%s[%d] = {%s};" % (name, T.ncol * T.ncol, ", ".join(str(float(x)) for row in T.color_num for x in row)))
    S("static cudaError_t launch_%s(int precision, const LaunchArgs& a) { return launch_multi(precision, a, parts_%s, %d, %d, color_num_%s); }"
      % (name, name, len(kernels), T.ncol, name))
    S("static size_t scratch_%s(int precision, long npad) { return multi_scratch_bytes(precision, npad, %d); }" % (name, T.ncol))
    algo = algorithmic_flops(T)
    S("extern const ProcTable tab_%s = {%d, %d, %d, %d, %d, %d, {%r, %r, %r}, {%r, %r, %r}, %r, color_num_%s, launch_%s, scratch_%s};"
      % (name, n, T.ndiagrams, total_namp, T.ncol, T.color_denom, len(kernels) + 1, float(algo), float(algo), float(algo),
         float(per_hel), float(per_hel), float(per_hel), float(fixed_max), name, name, name))
    S("}  // namespace me")
    files["gen_%s_table.cu" % name] = "\n".join(src) + "\n"
    info = dict(n=n, ndiagrams=T.ndiagrams, namp=total_namp, ncol=T.ncol, color_denom=T.color_denom,
                flops_per_helicity=algo, flops_executed_per_helicity=per_hel, fixed_flops=fixed_max, colour_flops=cs_flops, kernels=kinfo)
    return files, info
