"""Orbit-looped emitter for g g -> t t~ g g g (BASELINE.json config 5): 1240 diagrams, 1890 amplitude terms,
120 colour flows.  Same ideas as emit_orbit.py (shapes looped over gluon relabellings with table-driven
operands, two-sided quark line, bilinear / dual-current factorisations), plus what the size of the process forces:

  * the diagrams are split across THREE kernels (north_star: "splitting the diagrams across kernels": o0 the three-gluon
    sub-trees, o1 the 2+2 / 2+1 quark ends, o2 the four-gluon sub-trees made of pairs); every kernel loops over the helicities
    of the current chunk (ME_HEL_PER_CTA per CTA, grid.y over the chunk);
  * the 120 jamps do not fit on chip: each block instance accumulates the <= 36 colour flows it touches in
    per-thread shared-memory slots and adds them once into the global staging buffer gj[hel][flow][re/im][event]
    that the batched colour-sum kernel (csrc/color_sum.cu) contracts with the colour matrix.

Every diagram is cut at the gluon sub-tree that covers the third gluon along the quark line:
    amp = L . mid-slash . R,   L = row current with <= 2 gluons (from the t end), R = column current with <= 2
gluons (from the t~ end); (|L|,|mid|,|R|) = (0,5,0) 510, (0,4,1)+(1,4,0) 450, (0,3,2)+(2,3,0) 360, (1,3,1) 120,
(1,2,2)+(2,2,1) 180, (2,1,2) 270 amplitude terms = 1890.
"""
from itertools import permutations

from .emit import dd_invariant_lines, dd_k2, dd_q2
from .emit_orbit import Inst, FL, c_leaf, c_v3, c_v4, c_step, c_close, ONE, mask_of, SlotAlloc, eo, sum_expr
from .topology import color_matrix

N = 5
NPAR = 7
HEL_PER_CTA = 4  # helicities looped inside one CTA (csrc/multi.h ME_HEL_PER_CTA); the sharing kernels rely on the grouping of the list:
                 # entries 4 g .. 4 g + 3 share their gluon helicities (the four quark-helicity assignments, 255 = absent)
T_BIT, TB_BIT = NPAR - 1 - 2, NPAR - 1 - 3
# Measured and rejected variants are not kept as switches; what was tried and by how much it lost is in DESIGN.md section 8
# (a 256-thread CTA with a barrier per scope for kernel o0; a nested (u, w) loop in kernel o0; the tensor-memory layout for the FP32
# instantiations of o0 / o1; direct reductions instead of accumulators in kernel o2; accumulators instead of direct reductions in o1).
K1_PARTS = 1     # kernels the 18 closing vectors of the three-gluon sub-trees are spread over (1 as run; tests/test_abi_and_host.py
                 # checks with 2 and 3 that the algorithmic flop count does not depend on the split)
BLOCK1 = 128     # threads per CTA of every diagram kernel
FL5 = dict(FL, cx_comb=56, wadd=8, row_slash=64)
# FP64 kernels: categories kept in tensor memory so that two 128-thread CTAs fit per SM (8 warps instead of 4)
K1_UW_LOOP = False   # kernel o0: the two (u, w) halves of the closing vectors as a nested table-driven loop
K1_PRE = True        # sharing form o0s of kernel o0 (gluon-only currents of the three-gluon sub-trees once per group of helicities)
K1_CACHE_Q = (False, True)   # ... (FP64 form, FP32 form) with the one-gluon quark currents of a helicity in the current cache: one set per helicity
                             # instead of six rebuilds per block.  Measured per pass: FP32 40.8 against 41.5 ms; FP64 81.2 against 80.4 ms (the
                             # L2 latency of six more loads per block costs more than the 7 % of the arithmetic they save; through the L1: 81.8 ms)
K1S_UW_LOOP = True   # ... with the nested (u, w) loop in its FP64 form
TM_K1 = ("FERM", "TMP", "J")   # kernel o0: spinor bases, ubar / v / ubar gamma v, the parked current and 36 local jamp accumulators = 120 slots
TM_K2 = ("PAIR", "CHI")   # kernel o1: 10 gluon-pair currents + 5 column currents = 120 slots = 240 columns
K1_INIT_STAGING = (True, False)   # kernel o0 / o0s (FP64 forms: True) and o0f (FP32: False) zero the staging rows of a helicity themselves instead of a
                                  # memset in front of the pass.  Measured per pass: FP64 76.9 against 77.6 ms, FP32 40.3 against 40.1 ms.  (Plain stores on
                                  # the first touch of a row, chosen by a flag from the instance table, were slower: 78.9 ms, the flush code doubles.)
K2_CACHE_COLS = True     # kernel o1: the two column currents of every gluon pair parked in the current cache by the cols2 loop and reloaded by rows2
MIN_CTAS_F32 = {"2s": 3}  # kernel tag -> minimum CTAs per SM asked of the compiler for the FP32 instantiation (register cap).  o2s in FP32 is latency-bound and
                          # small in shared / tensor memory: 168 registers (8 B of spill) and three CTAs per SM: FP32 pass 40.1 -> 39.2 ms; four (128 registers): 40.4 ms
K3S_CACHE_U = True       # sharing kernel o2s: the thirty ordered currents of a group in the L2-resident current cache (two CTAs per SM) instead of on chip (one)
K3D_JACC = 48            # accumulator kernel o2d (current sharing off): one set of local jamp accumulators per last gluon, kept in tensor memory
TM_K3 = ("J",)            # FP64: 96 slots = 192 columns, one CTA per SM; FP32: one column per slot, two CTAs per SM


class Layout5:
    """per-thread shared-memory slots of one kernel (units of R), paired layout of hel_amp.cuh"""
    npar = NPAR

    def __init__(self, want_pairs, want_iq_mid, jacc, ferm_smem=False, want_q1chi=True, want_chi=False, ik2_sizes=(2, 3, 4, 5), scratch=False, tm=(), jtt4=False, nu=0, nu_smem=0):
        # tm: categories ("PAIR", "CHI") that the FP64 kernel keeps in tensor memory (hel_amp.cuh "Tensor memory as a per-thread
        # scratchpad"); they are allocated last, from the even slot TM0 on, so that the shared-memory part is contiguous
        A = SlotAlloc()
        self.FERM = None
        if ferm_smem and "FERM" not in tm:    # ubar, v, ubar gamma v of the current helicity + the two spinor bases
            self.FERM = dict(ub=A.vec(8), vv=A.vec(8), jtt=A.vec(8), sbt=A.vec(5), sbtb=A.vec(5))
        self.MOM = A.vec(4 * N)
        self.PT = A.vec(4)
        self.GBS = [A.vec(5) for _ in range(N)]
        self.JTT4 = A.vec(8 * HEL_PER_CTA) if jtt4 else None      # ubar gamma v of the helicities of the CTA's group (sharing kernel o2s)
        # colour-ordered currents of the sharing kernel o2s: U[(w, k)], the first nu_smem of every w in shared memory, the rest in TMEM
        self.U = {(w, k): A.vec(8) for w in range(N) for k in range(nu_smem)}
        self.PAIR = {}
        pairs = [(a, b) for a in range(N) for b in range(a + 1, N)]
        if want_pairs and "PAIR" not in tm:
            self.PAIR = {p: A.vec(8) for p in pairs}
        self.Q1 = self.CHI = None             # one-gluon currents of both quark ends (kernel 1 rebuilds them at each use instead)
        if want_q1chi:
            assert "CHI" not in tm
            self.Q1 = A.vec(8 * N)
            self.CHI = A.vec(8 * N)
        elif want_chi and "CHI" not in tm:
            self.CHI = A.vec(8 * N)
        self.TMP = A.vec(8) if (scratch and "TMP" not in tm) else None   # one parked current (kernel 1)
        if "J" not in tm:
            self.J = A.vec(2 * jacc)
        self.jacc = jacc
        masks2 = [m for m in range(1, 1 << N) if bin(m).count("1") in ik2_sizes]
        self.IK2 = {m: A.scalar() for m in masks2}
        # quark propagators: row side sets of size 1,2 and (for the column currents) size 3,4
        masksq = [m for m in range(1, (1 << N) - 1) if want_iq_mid or bin(m).count("1") in (1, 4)]
        self.IQ = {m: A.scalar() for m in masksq}
        if tm:
            self.TM0 = A.vec(0)
            if ferm_smem and "FERM" in tm:            # the spinor bases take a whole 8-slot vector each in TMEM (one tcgen05 x16 access)
                self.FERM = dict(sbt=A.vec(8), sbtb=A.vec(8), ub=A.vec(8), vv=A.vec(8), jtt=A.vec(8))
            if scratch and "TMP" in tm:
                self.TMP = A.vec(8)
            if want_pairs and "PAIR" in tm:
                self.PAIR = {p: A.vec(8) for p in pairs}
            if want_chi and "CHI" in tm:
                self.CHI = A.vec(8 * N)
            if "J" in tm:
                assert jacc % 4 == 0
                self.J = A.vec(2 * jacc)
            if "U" in tm:
                self.U.update({(w, k): A.vec(8) for w in range(N) for k in range(nu_smem, nu)})
            self.tm_cols = 32
            while self.tm_cols < 2 * (A.n - self.TM0):
                self.tm_cols *= 2                      # tcgen05.alloc takes a power of two >= 32
            assert self.tm_cols <= 512, (self.TM0, self.tm_cols)      # 256 columns and 113 slots: two CTAs per SM
        self.nslots = A.n + (A.n & 1)


class Inst5(Inst):
    """Block instance whose jamps go to LOCAL accumulators (shared memory) and are flushed to global staging."""

    def __init__(self, lay, stride, inner=False, parent=None):
        super().__init__(lay, stride)
        self.subtables = []          # (name, [param rows]) of nested loops
        self.parent = parent         # inner instance that accumulates into the local jamp slots of its outer instance
        if inner:                    # body of a nested loop: own table row `tb2`, may use the variables of the outer instance
            self.tbname = "tb2"
        self.local = {}              # global colour-flow index -> local accumulator slot
        self.redundant = 0           # flops that recompute something another block / kernel also computes
        self.scopes = [set()]        # names of fermion values loaded in each open brace scope

    def L(self, s):
        super().L(s)
        for ch in s:
            if ch == "{":
                self.scopes.append(set())
            elif ch == "}":
                self.scopes.pop()

    def fv(self, *names):
        """make ub / vv / jtt usable here: registers of the kernel scope, or (kernels that keep them in shared
        memory to relieve register pressure) loaded into the current brace scope"""
        if self.lay.FERM is None:
            return
        for name in names:
            if any(name in sc for sc in self.scopes):
                continue
            if self.in_tm(self.lay.FERM[name]):
                self.L("XW<R, TM> %s_x; xldw_issue<R, TM>(%s_x, sm, tm, %d);" % (name, name, eo(self.lay.FERM[name], self.stride)))
                self.L("const W4<R> %s = xldw_get<R, TM>(%s_x);" % (name, name))
            else:
                self.L("const W4<R> %s = ldw<R>(sm + %d);" % (name, eo(self.lay.FERM[name], self.stride)))
            self.scopes[-1].add(name)

    def flush_jamps(self):
        ups = []
        for sigma, u, z in self.grouped_updates():
            owner = self.parent if self.parent is not None else self
            loc = owner.local.setdefault(sigma, len(owner.local))
            assert loc < self.lay.jacc, "local jamp accumulators exhausted"
            re, im = self.unit_times(u, z)
            o = eo(self.lay.J + 2 * loc, self.stride)
            # the slot of a flow differs between the iterations of a nested loop: table-driven there, immediate otherwise
            ups.append((self.P(o) if self.parent is not None else "%d" % o, re, im))
            self.flops += 2
        self.emit_accumulate(ups)

    RED_BATCH = 8

    def flush_direct(self):
        """pending jamp updates go straight into the global staging buffer, one fire-and-forget reduction per colour flow
        (all amplitudes that feed a flow are combined in registers first).  For blocks in which a flow is touched once: a
        shared-memory accumulator there is a read-modify-write plus a flush for nothing."""
        ups = self.grouped_updates()
        # the row offsets come from the instance table (indexed constant loads, long latency) and feed integer address arithmetic:
        # they are formed in batches ahead of the reductions that use them, so that the loads of a batch are in flight together
        for b0 in range(0, len(ups), self.RED_BATCH):
            batch = ups[b0:b0 + self.RED_BATCH]
            self.L("{ const unsigned " + ", ".join("ro%d = (unsigned)%s * npad32" % (i, self.P(2 * sigma)) for i, (sigma, u, z) in enumerate(batch)) + ";")
            for i, (sigma, u, z) in enumerate(batch):
                re, im = self.unit_times(u, z)
                self.L("  { RJ* g = gj + ro%d; atomicAdd(g, (RJ)(%s)); atomicAdd(g + npad32, (RJ)(%s)); }" % (i, re, im))
                self.flops += 2
            self.L("}")

    def inner_loop(self, name, inners):
        """nested table-driven loop over `inners` (Inst5(inner=True) objects of identical shape) inside this instance"""
        t = inners[0]
        for it in inners[1:]:
            assert it.lines == t.lines and it.jamp_codes == t.jamp_codes, "inner instances of %s differ" % name
        self.L("#pragma unroll 1")
        self.L("for (int i2 = 0; i2 < %d; ++i2) {" % len(inners))
        self.L("  const int* tb2 = &@SUB:%s@[it * %d + i2][0];" % (name, len(inners)))
        for l in t.lines:
            self.L("  " + l)
        self.L("}")
        self.subtables.append((name, [it.params for it in inners]))
        self.flops += sum(it.flops for it in inners)
        self.namp += sum(it.namp for it in inners)
        self.redundant += sum(it.redundant for it in inners)
        self.jamp_codes.extend(t.jamp_codes)

    def flush_global(self):
        """add the local accumulators into gj and clear them.  The add is a fire-and-forget reduction (RED.ADD, no
        read latency); every address is private to one thread, whose program order fixes the order of the adds, so
        the result is deterministic run to run."""
        def out(sigma, re, im):
            return "{ RJ* g = gj + (unsigned)%s * npad32; atomicAdd(g, (RJ)%s); atomicAdd(g + npad32, (RJ)%s); }" % (self.P(2 * sigma), re, im)
        if self.in_tm(self.lay.J):
            # accumulators in tensor memory: four flows per tcgen05.ld x16, reduced into gj, cleared with one tcgen05.st x16
            items = sorted(self.local.items(), key=lambda t: t[1])
            assert [loc for _, loc in items] == list(range(len(items)))
            self.L("xwait_st<TM>();")
            for g0 in range(0, len(items), 4):
                grp = items[g0:g0 + 4]
                o = eo(self.lay.J + 2 * g0, self.stride)
                self.L("{ XW<R, TM> jx; xldw_issue<R, TM>(jx, sm, tm, %d);" % o)
                self.L("  const W4<R> jw = xldw_get<R, TM>(jx);")
                for k, (sigma, loc) in enumerate(grp):
                    self.L("  " + out(sigma, "jw.r%d" % k, "jw.i%d" % k))
                    self.flops += 2; self.redundant += 2
                self.L("  xstw<R, TM>(sm, tm, %d, W4<R>{(R)0, (R)0, (R)0, (R)0, (R)0, (R)0, (R)0, (R)0}); }" % o)
            self.local = {}
            return
        for sigma, loc in sorted(self.local.items(), key=lambda t: t[1]):
            o = eo(self.lay.J + 2 * loc, self.stride)
            self.L(out(sigma, "sm[%d]" % o, "sm[%d]" % (o + 1)))
            self.L("sm[%d] = 0; sm[%d] = 0;" % (o, o + 1))
            self.flops += 2; self.redundant += 2     # staging adds are overhead of the multi-kernel split, not of the method
        self.local = {}


def _cdiff(A, B, C):
    """colour polynomial A - (B - C); empty when the colour-ordering identity A = B - C holds"""
    out = dict(A)
    for P, k in ((B, -1), (C, 1)):
        for st, v in P.items():
            out[st] = out.get(st, 0) + k * v
    return {st: v for st, v in out.items() if abs(v) > 1e-12}


def cpair(a, b):
    return c_v3(c_leaf(a), c_leaf(b))


def cq1(l):
    return c_step(ONE, c_leaf(l))


def cchi(l):
    return c_step(c_leaf(l), ONE)


def rest_of(*labels):
    return [l for l in range(N) if l not in labels]


def full_mask():
    return (1 << N) - 1


# ------------------------------------------------------------------------------------------
# shared code fragments
# ------------------------------------------------------------------------------------------
def emit_pair(I, name, a, b, ea, eb, ka, kb):
    I.L("const W4<R> %s = v3_current(%s, %s, %s, %s, %s);" % (name, ea, eb, ka, kb, I.ik2(a, b)))
    I.flops += FL5["v3_current"]


def emit_rows2(I, a, b, pab, ea, eb):
    """the two colour-ordered row currents with gluons {a,b} attached (a<b): returns [(name, colour)]"""
    if I.lay.Q1 is not None:
        I.ldw("q1a", I.lay.Q1 + 8 * a); I.ldw("q1b", I.lay.Q1 + 8 * b)
    else:                                 # no Q1 slots: the two one-gluon row currents are formed here
        f0 = I.flops
        I.qvec("qa1", [a]); I.qvec("qb1", [b]); I.fv("ub")
        I.L("const W4<R> q1a = quark_step2(ub, %s, qa1, mt, %s), q1b = quark_step2(ub, %s, qb1, mt, %s);" % (ea, I.iq(a), eb, I.iq(b)))
        I.flops += 2 * FL5["quark_step2"]; I.redundant += I.flops - f0
    I.qvec("qr", [a, b])
    I.L("const R iqr = %s;" % I.iq(a, b))
    I.fv("ub")
    # colour-ordered form: the pair current (a commutator, colour ab - ba) is folded into the two stepwise currents in
    # front of their common propagator: two currents, one colour string each, instead of three
    col_ab, col_ba = c_step(cq1(a), c_leaf(b)), c_step(cq1(b), c_leaf(a))
    assert not _cdiff(c_step(ONE, cpair(a, b)), col_ab, col_ba)
    I.L("const W4<R> spr = row_slash(ub, %s);" % pab)
    I.L("const W4<R> rb = row_step(wadd(row_slash(q1a, %s), spr), qr, mt, iqr), rc = row_step(wsub(row_slash(q1b, %s), spr), qr, mt, iqr);" % (eb, ea))
    I.flops += 3 * FL5["row_slash"] + 2 * (FL5["wadd"] + FL5["col_step"])
    return [("rb", col_ab), ("rc", col_ba)]


def emit_cols2(I, c, d, pcd, ec, ed, tag="", cached=None):
    """the two colour-ordered column currents with gluons {c,d} attached (c<d), grown from the t~ end; cached = first vector of the
    pair in the current cache: the currents are loaded from there (the cols2 loop of the same helicity has parked them) instead of built"""
    col_cd, col_dc = c_step(c_leaf(c), cchi(d)), c_step(c_leaf(d), cchi(c))
    if cached is not None:
        vec = I.P(cached)
        I.L("const W4<R> cb%s = sc_ldw<R>(sc, %s), cc%s = sc_ldw<R>(sc, %s + 1);" % (tag, vec, tag, vec))
        return [("cb" + tag, col_cd), ("cc" + tag, col_dc)]
    I.ldw("chc" + tag, I.lay.CHI + 8 * c); I.ldw("chd" + tag, I.lay.CHI + 8 * d)
    row_side = rest_of(c, d)
    I.qvec("qc" + tag, row_side)
    I.L("const R iqc%s = %s;" % (tag, I.iq(*row_side)))
    I.fv("vv")
    # colour of a column step: -(gluon)(previous column); colour-ordered as in emit_rows2
    assert not _cdiff(c_step(cpair(c, d), ONE), col_cd, col_dc)
    I.L("const W4<R> spc%s = slash_col(%s, vv);" % (tag, pcd))
    I.L("const W4<R> cb%s = col_step(wadd(slash_col(%s, chd%s), spc%s), qc%s, mt, iqc%s), cc%s = col_step(wsub(slash_col(%s, chc%s), spc%s), qc%s, mt, iqc%s);"
        % (tag, ec, tag, tag, tag, tag, tag, ed, tag, tag, tag, tag))
    I.flops += 3 * FL5["slash_col"] + 2 * (FL5["wadd"] + FL5["col_step"])
    return [("cb" + tag, col_cd), ("cc" + tag, col_dc)]


def phase_a(lay, stride, add_group, want_pairs):
    labels = list(range(N))
    if want_pairs:
        insts = []
        for (a, b) in lay.PAIR:
            I = Inst5(lay, stride)
            I.leaf("ea", a); I.leaf("eb", b); I.kvec("ka", [a]); I.kvec("kb", [b])
            emit_pair(I, "t", a, b, "ea", "eb", "ka", "kb")
            I.stw(lay.PAIR[(a, b)], "t")
            insts.append(I)
        add_group("pairs", insts, 2)
    if lay.CHI is None:
        return
    if lay.Q1 is not None:
        insts = []
        for l in labels:
            I = Inst5(lay, stride)
            I.leaf("el", l); I.qvec("q", [l]); I.fv("ub")
            I.L("const W4<R> t = quark_step2(ub, el, q, mt, %s);" % I.iq(l)); I.flops += FL5["quark_step2"]
            I.stw(lay.Q1 + 8 * l, "t")
            insts.append(I)
        add_group("q1", insts, 1)
    insts = []
    for w in labels:
        rest = rest_of(w)
        I = Inst5(lay, stride)
        I.leaf("ew", w); I.qvec("q", rest); I.fv("vv")
        I.L("const W4<R> t = col_step(slash_col(ew, vv), q, mt, %s);" % I.iq(*rest)); I.flops += FL5["slash_col"] + FL5["col_step"]
        I.stw(lay.CHI + 8 * w, "t")
        insts.append(I)
    add_group("chi1", insts, 1)


# ------------------------------------------------------------------------------------------
# kernel 1: everything that contains a three-gluon sub-tree t on M = {a,b,c}; {x,y} = the other two gluons.
# The 6 terms t_i stay in registers; 18 four-vectors X_j (bilinears of the fermion ends, dual currents of the
# vertices that would extend t) are formed one after the other and each gives 6 amplitudes t_i . X_j.
# ------------------------------------------------------------------------------------------
def build_k1(stride, pidx, part=None, nparts=3, uw_loop=None, pre=False, cache_q=False, init_staging=False):
    """part = None: all 18 vectors in one kernel; part = 0,1,2: six vectors each (the kernel then fits the
    instruction cache: the single kernel was ~12.5 k SASS instructions and stalled on instruction fetch)"""
    # no Q1 / CHI slots: the one-gluon quark currents are rebuilt where they are used (12 per block, ~15 % more flops), which
    # brings the kernel from 292 to 220 slots per thread (incl. one scratch vector that carries chi1(w) / q1(u) across scopes), i.e. from 96 to 128 threads per CTA (all four schedulers busy)
    lay = Layout5(want_pairs=False, want_iq_mid=True, jacc=36, ferm_smem=True, want_q1chi=False, scratch=True, tm=TM_K1)
    groups = []
    add_group = _grouper(groups)
    phase_a(lay, stride, add_group, want_pairs=False)
    QV, CV = 30, 35             # current cache, sharing form: vectors 0..29 per group (three per block), 30..34 q1(l), 35..39 chi1(w) per helicity
    if cache_q and pre:
        qi, ci = [], []
        for l in range(N):
            I = Inst5(lay, stride)
            I.leaf("el", l); I.qvec("q", [l]); I.fv("ub")
            I.L("const W4<R> t = quark_step2(ub, el, q, mt, %s);" % I.iq(l)); I.flops += FL5["quark_step2"]
            I.L("sc_stw<R>(sc, %s, t);" % I.P(QV + l))
            I.redundant += I.flops       # the algorithmic count has one set of one-gluon quark currents already (kernel o1 / the q1 reference loop)
            qi.append(I)
            rest = rest_of(l)
            I = Inst5(lay, stride)
            I.leaf("ew", l); I.qvec("q", rest); I.fv("vv")
            I.L("const W4<R> t = col_step(slash_col(ew, vv), q, mt, %s);" % I.iq(*rest)); I.flops += FL5["slash_col"] + FL5["col_step"]
            I.L("sc_stw<R>(sc, %s, t);" % I.P(CV + l))
            I.redundant += I.flops
            ci.append(I)
        add_group("q1c", qi, 1)
        add_group("chi1c", ci, 1)
    insts, pre_insts = [], []
    for vi, M in enumerate([(a, b, c) for a in range(N) for b in range(a + 1, N) for c in range(b + 1, N)]):
        a, b, c = M
        x, y = rest_of(a, b, c)
        I = Inst5(lay, stride)
        I.leaf("ex", x); I.leaf("ey", y); I.kvec("kx", [x]); I.kvec("ky", [y])
        I.L("const R ik5 = %s;" % I.ik2(*range(N)))
        # pre: the two ordered currents of the sub-tree and the pair current of the other two gluons depend on the gluon helicities
        # only: the sharing form of the kernel builds them once per group of helicities (G) and parks them in the L2-resident
        # current cache (vectors 3 vi .. 3 vi + 2); the block reloads them
        G = Inst5(lay, stride) if pre else I
        if pre:
            G.L("W4<R> pxy;")
            G.L("{")
            G.leaf("ex", x); G.leaf("ey", y); G.kvec("kx", [x]); G.kvec("ky", [y])
            G.L("const W4<R> t = v3_current(ex, ey, kx, ky, %s); pxy = t;" % G.ik2(x, y)); G.flops += FL5["v3_current"]
            G.L("}")
            I.L("const W4<R> pxy = sc_ldw<R>(sc, %s + 2);" % I.P(3 * vi))
        else:
            emit_pair(I, "pxy", x, y, "ex", "ey", "kx", "ky")
        # the six three-gluon terms on M (registers for the whole block); their inputs die in this scope
        tcol = [c_v3(cpair(a, b), c_leaf(c)), c_v3(cpair(a, c), c_leaf(b)), c_v3(cpair(b, c), c_leaf(a))] + \
               [c_v4(k, c_leaf(a), c_leaf(b), c_leaf(c)) for k in range(3)]
        # colour-ordered form of the three-gluon sub-tree: the four-gluon-vertex pieces carry the colours of the three
        # channels, and the Jacobi identity col1 = col0 + col2 leaves two independent currents instead of six terms
        assert all(not _cdiff(tcol[3 + k], tcol[k], {}) for k in range(3)) and not _cdiff(tcol[1], tcol[0], {st: -v for st, v in tcol[2].items()})
        tnames, tcol = ["s0", "s2"], [tcol[0], tcol[2]]
        I.L("W4<R> s0, s2; P4<R> kM;")
        if pre:
            G.L("W4<R> s0, s2;")
        G.L("{")
        for nm, l in (("ea", a), ("eb", b), ("ec", c)):
            G.leaf(nm, l)
        for nm, l in (("ka", a), ("kb", b), ("kc", c)):
            G.kvec(nm, [l])
        G.L("const P4<R> kab = padd(ka, kb), kac = padd(ka, kc), kbc = padd(kb, kc);"); G.flops += 12
        if not pre:
            I.L("kM = padd(kab, kc);"); I.flops += 4
        emit_pair(G, "pab", a, b, "ea", "eb", "ka", "kb"); emit_pair(G, "pac", a, c, "ea", "ec", "ka", "kc")
        emit_pair(G, "pbc", b, c, "eb", "ec", "kb", "kc")
        G.redundant += 3 * FL5["v3_current"]          # every pair is formed in 4 blocks; once (as pxy of its own block) would do
        G.L("const R ik3 = %s;" % G.ik2(a, b, c))
        G.L("const V4Dots<R> dots = v4_dots(ea, eb, ec, ik3);"); G.flops += FL5["v4_dots"]
        G.L("const W4<R> t14 = wadd(v3_current(pac, eb, kac, kb, ik3), v4_current(1, dots, ea, eb, ec));")
        G.L("s0 = wadd(wadd(v3_current(pab, ec, kab, kc, ik3), v4_current(0, dots, ea, eb, ec)), t14);")
        G.L("s2 = wadd(wadd(v3_current(pbc, ea, kbc, ka, ik3), v4_current(2, dots, ea, eb, ec)), t14);")
        G.flops += 5 * FL5["wadd"] + 3 * FL5["v3_current"] + 3 * FL5["v4_current"]
        G.L("}")
        if pre:
            vec = G.P(3 * vi)
            G.L("sc_stw<R>(sc, %s, s0); sc_stw<R>(sc, %s + 1, s2); sc_stw<R>(sc, %s + 2, pxy);" % (vec, vec, vec))
            pre_insts.append(G)
            vec = I.P(3 * vi)
            I.L("s0 = sc_ldw<R>(sc, %s); s2 = sc_ldw<R>(sc, %s + 1);" % (vec, vec))
            I.L("{")
            for nm, l in (("ka", a), ("kb", b), ("kc", c)):
                I.kvec(nm, [l])
            I.L("kM = padd(padd(ka, kb), kc);"); I.flops += 8
            I.L("}")
        if part is not None and part > 0:             # the split kernels each rebuild pxy and the six terms: all of it overhead
            I.redundant = I.flops

        counter = [0]

        def dots_with(T, prelude, xexpr, flops, colour_of_term, post=None):
            """6 amplitudes t_i . X and their jamp updates, emitted into instance T (the block, or the body of its nested
            (u, w) loop); operands of X are loaded inside the scope"""
            idx = counter[0]; counter[0] += 1
            if part is not None and idx // (18 // nparts) != part:
                return
            T.L("{ if (sizeof(R) == 8) ME_FENCE;")      # FP64 only: stops load hoisting that would spill
            for fn in prelude:
                fn(T)
            T.fv(*[nm for nm in ("ub", "vv", "jtt") if nm in xexpr])
            T.L("  const W4<R> X = %s;" % xexpr); T.flops += flops
            if post is not None:
                post(T)
            T.L("  const Cx<R> " + ", ".join("a%d = wdot(%s, X)" % (k, tn) for k, tn in enumerate(tnames)) + ";")
            T.flops += len(tnames) * FL5["wdot"]
            T.namp += 6 - len(tnames)                # diagram terms folded into the colour-ordered currents
            for i, col in enumerate(tcol):
                T.jamp("a%d" % i, colour_of_term(col), pidx)
            T.flush_jamps()
            T.L("}")

        def mk_q1(nm, l, el):
            """q1(l) = ubar with gluon l attached (polarisation vector el), rebuilt in the current scope"""
            def f(T):
                f0 = T.flops
                T.qvec("qk_" + nm, [l]); T.fv("ub")
                T.L("const W4<R> %s = quark_step2(ub, %s, qk_%s, mt, %s);" % (nm, el, nm, T.iq(l)))
                T.flops += FL5["quark_step2"]; T.redundant += T.flops - f0
            return f

        def mk_chi(nm, w, ew):
            """chi1(w) = v with gluon w attached (polarisation vector ew), rebuilt in the current scope"""
            def f(T):
                rest = rest_of(w)
                f0 = T.flops
                T.qvec("qk_" + nm, rest); T.fv("vv")
                T.L("const W4<R> %s = col_step(slash_col(%s, vv), qk_%s, mt, %s);" % (nm, ew, nm, T.iq(*rest)))
                T.flops += FL5["slash_col"] + FL5["col_step"]; T.redundant += T.flops - f0
            return f

        row_side = rest_of(x, y)
        qc = lambda T: (T.qvec("qc", row_side), T.L("const R iqc = %s;" % T.iq(*row_side)))
        qr = lambda T: (T.qvec("qr", [x, y]), T.L("const R iqr = %s;" % T.iq(x, y)))
        stc = FL5["slash_col"] + FL5["col_step"] + FL5["bilinear"]
        str_ = FL5["quark_step2"] + FL5["bilinear"]

        def uw_vectors(T, u, w, eu, ew, ku, kw):
            """the six closing vectors that come in a (u, w) = (x, y), (y, x) pair"""
            quad = lambda col: c_v3(col, c_leaf(u))
            ik4 = lambda T_: T_.L("const R ik4 = %s;" % T_.ik2(a, b, c, u))
            # chi1(w) is formed once and parked in the scratch vector for its three scopes; q1(u) takes the slot over for its second
            park = lambda nm: (lambda T_: T_.stw(lay.TMP, nm))
            fetch = lambda nm: (lambda T_: T_.ldw(nm, lay.TMP))
            # quad = V3(t, eps_u) closing three ways with the last gluon w: on the t~ end (colour Q.w), on the t end (w.Q), or through a
            # three-gluon vertex on the bare line (colour Q.w - w.Q): the current of the third, y3, is folded into the other two
            # (two scopes instead of three)
            y3 = lambda T_: (T_.fv("jtt"), T_.L("const W4<R> y3 = v3_dual(%s, jtt, padd(kM, %s), %s, ik5);" % (ew, ku, kw)))
            if cache_q and pre:
                # sharing form: the one-gluon quark currents come from the current cache (formed once per helicity by the q1c / chi1c loops
                # instead of six times per block), which leaves the scratch vector to y3 (formed once instead of twice)
                cached = lambda nm, base, l: (lambda T_: T_.L("const W4<R> %s = sc_ldw<R>(sc, %s);" % (nm, T_.P(base + l))))
                get_chw, get_q1w, get_q1u, get_q1u2 = cached("chw", CV, w), cached("q1w", QV, w), cached("q1u", QV, u), cached("q1u", QV, u)
                y3a = lambda T_: (y3(T_), park("y3")(T_)); y3b = fetch("y3")
                post_q1u = None
            else:
                T.L("{"); mk_chi("chw", w, ew)(T); park("chw")(T); T.L("}")
                get_chw, get_q1w, get_q1u, get_q1u2 = fetch("chw"), mk_q1("q1w", w, ew), mk_q1("q1u", u, eu), fetch("q1u")
                y3a = y3b = y3
                post_q1u = park("q1u")
            dots_with(T, [get_chw, ik4, y3a], "v3_dual(%s, wadd(bilinear(ub, chw), y3), kM, %s, ik4)" % (eu, ku),
                      2 * FL5["v3_dual"] + FL5["bilinear"] + FL5["wadd"] + 4, lambda col: c_close(ONE, quad(col), cchi(w)))
            dots_with(T, [get_q1w, ik4, y3b], "v3_dual(%s, wsub(bilinear(q1w, vv), y3), kM, %s, ik4)" % (eu, ku),
                      (2 if y3b is y3 else 1) * FL5["v3_dual"] + FL5["bilinear"] + FL5["wadd"] + (4 if y3b is y3 else 0), lambda col: c_close(cq1(w), quad(col), ONE))
            idx3 = counter[0]; counter[0] += 1
            if part is None or idx3 // (18 // nparts) == part:
                T.namp += 6                   # the six V3-closing terms are inside the twelve above
            if (part is None or (idx3 - 1) // (18 // nparts) == part) and y3b is y3:
                T.redundant += FL5["v3_dual"] + 4  # y3 is formed twice
            # ubar . t-slash . chi2: eps_u attached to chi1(w)
            dots_with(T, [qc, get_chw], "bilinear(ub, col_step(slash_col(%s, chw), qc, mt, iqc))" % eu, stc,
                      lambda col: c_close(ONE, col, c_step(c_leaf(u), cchi(w))))
            # q1(u) . t-slash . chi1(w)
            dots_with(T, [get_q1u, get_chw], "bilinear(q1u, chw)", FL5["bilinear"], lambda col: c_close(cq1(u), col, cchi(w)),
                      post=post_q1u)
            # q2 . t-slash . v: eps_w attached to q1(u)
            dots_with(T, [qr, get_q1u2], "bilinear(quark_step2(q1u, %s, qr, mt, iqr), vv)" % ew, str_,
                      lambda col: c_close(c_step(cq1(u), c_leaf(w)), col, ONE))

        if K1_UW_LOOP if uw_loop is None else uw_loop:
            # one nested table-driven loop of two iterations instead of two copies of five scopes; its jamp updates go to the
            # block's accumulators (slots from the table)
            inners = []
            for (u, w) in ((x, y), (y, x)):
                J = Inst5(lay, stride, inner=True, parent=I)
                J.leaf("eu", u); J.leaf("ew", w); J.kvec("ku", [u]); J.kvec("kw", [w])
                J.redundant += J.flops                # ex, ey, kx, ky exist in the block
                uw_vectors(J, u, w, "eu", "ew", "ku", "kw")
                inners.append(J)
            I.inner_loop("uw", inners)
        else:
            uw_vectors(I, x, y, "ex", "ey", "kx", "ky")
            uw_vectors(I, y, x, "ey", "ex", "ky", "kx")
        # V3(t, pair(x,y)) on the bare line
        dots_with(I, [], "v3_dual(pxy, jtt, kM, padd(kx, ky), ik5)", FL5["v3_dual"] + 4, lambda col: c_close(ONE, c_v3(col, cpair(x, y)), ONE))
        # V4(t, eps_x, eps_y) on the bare line, three structures (duals of the contact term)
        cdots = lambda T: (T.fv("jtt"), T.L("const Cx<R> cxj = cxs(wdot(ex, jtt), ik5), cyj = cxs(wdot(ey, jtt), ik5), cxy = cxs(wdot(ex, ey), ik5);"))
        dots_with(I, [cdots], "cx_comb(cxj, ey, cxy, jtt)", FL5["cx_comb"] + 3 * FL5["wdot"] + 6, lambda col: c_close(ONE, c_v4(0, col, c_leaf(x), c_leaf(y)), ONE))
        dots_with(I, [cdots], "cx_comb(cyj, ex, cxy, jtt)", FL5["cx_comb"], lambda col: c_close(ONE, c_v4(1, col, c_leaf(x), c_leaf(y)), ONE))
        dots_with(I, [cdots], "cx_comb(cyj, ex, cxj, ey)", FL5["cx_comb"], lambda col: c_close(ONE, c_v4(2, col, c_leaf(x), c_leaf(y)), ONE))
        # ubar . t-slash . chi2(pair)  and  q2(pair) . t-slash . v
        # (one current at a time: three live two-gluon currents next to t0..t5 would spill)
        dots_with(I, [qc], "bilinear(ub, col_step(slash_col(pxy, vv), qc, mt, iqc))", stc, lambda col: c_close(ONE, col, c_step(cpair(x, y), ONE)))
        dots_with(I, [qr], "bilinear(quark_step2(ub, pxy, qr, mt, iqr), vv)", str_, lambda col: c_close(c_step(ONE, cpair(x, y)), col, ONE))
        assert counter[0] == 18
        I.flush_global()
        insts.append(I)
    if pre:
        add_group("tripre", pre_insts, 1)
        t = groups[-1][1]
        t.pre = True                      # run once per group of helicities, before the helicity loop
        t.group_flops = t.flops; t.flops = 0
        t.group_redundant = t.redundant; t.redundant = 0
        t.cache_vectors = 3 * len(pre_insts) + (10 if cache_q else 0)
    add_group("triples", insts, 1)
    # the first kernel of a pass can zero the staging rows of a helicity itself, right before it adds into them (the lines are then in the L2
    # for its first reductions), instead of a memset of the whole chunk in front of the pass
    groups[-1][1].init_staging = bool(init_staging) and (part is None or part == 0)
    return lay, groups


def _grouper(groups):
    def add_group(name, insts, unroll=1):
        tmpl = insts[0]
        for it in insts[1:]:
            assert it.lines == tmpl.lines, "instances of %s differ in shape" % name
            assert it.jamp_codes == tmpl.jamp_codes, "instances of %s differ in colour coefficients" % name
        groups.append((name, tmpl, [it.params for it in insts], unroll))
        for si, (sname, _) in enumerate(tmpl.subtables):
            tmpl.subtables[si] = (sname, [r for it in insts for r in it.subtables[si][1]])
    return add_group


def spair(p):
    return tuple(sorted(p))


# ------------------------------------------------------------------------------------------
# kernel 2: amplitudes whose two ends carry (2 | 2), (2 | 1) or (1 | 2) gluons and whose middle is a gluon or a pair
# ------------------------------------------------------------------------------------------
def build_k2(stride, pidx, cache_cols=None):
    cache_cols = K2_CACHE_COLS if cache_cols is None else cache_cols
    # 226 slots per thread -> 128 threads per CTA: no Q1 slots (the row-side one-gluon currents are formed where they are
    # used: 5 per ten uses would do, +14 % flops), only the pair propagators; no local jamp accumulators: every (sub-)block touches each
    # colour flow once, its amplitudes are combined per flow in registers and added straight into the staging buffer
    lay = Layout5(want_pairs=True, want_iq_mid=True, jacc=0, want_q1chi=False, want_chi=True, ik2_sizes=(2,), tm=TM_K2)
    groups = []
    add_group = _grouper(groups)
    phase_a(lay, stride, add_group, want_pairs=True)
    pair_index = {p_: i_ for i_, p_ in enumerate(lay.PAIR)}
    # ---- rows2 loop: A = {a,b}; the three row currents on A meet (i) eps_m . chi2(B), (ii) pair(P) . chi1(w)
    insts = []
    for (a, b) in lay.PAIR:
        rest = rest_of(a, b)
        I = Inst5(lay, stride)
        I.leaf("ea", a); I.leaf("eb", b)
        I.ldw("pab", lay.PAIR[(a, b)])
        rows = emit_rows2(I, a, b, "pab", "ea", "eb")
        for i, m in enumerate(rest):
            c, d = [l for l in rest if l != m]
            t = "_%d" % i
            I.L("{")
            I.leaf("em", m); I.leaf("ec", c); I.leaf("ed", d)
            I.ldw("pcd", lay.PAIR[(c, d)])
            f0 = I.flops
            cols = emit_cols2(I, c, d, "pcd", "ec", "ed", cached=2 * pair_index[(c, d)] if cache_cols else None)
            I.redundant += I.flops - f0                 # the cols2 loop forms the same two currents of the pair (c, d): needed once per helicity
            I.namp += (9 - len(rows) * len(cols)) + (3 - len(rows))     # diagram terms folded into the colour-ordered currents
            xs = ["x%d" % k for k in range(len(cols))]
            I.L("const W4<R> " + ", ".join("%s = slash_col(em, %s)" % (xn, cn) for xn, (cn, _) in zip(xs, cols)) + ";"); I.flops += len(cols) * FL5["slash_col"]
            for ri, (rn, rcol) in enumerate(rows):       # the amplitudes of this sub-block are combined per colour flow and added once
                I.L("const Cx<R> " + ", ".join("a%d_%d = row_col(%s, %s)" % (k, ri, rn, xn) for k, xn in enumerate(xs)) + ";"); I.flops += len(xs) * FL5["row_col"]
                for k, (cn, ccol) in enumerate(cols):
                    I.jamp("a%d_%d" % (k, ri), c_close(rcol, c_leaf(m), ccol), pidx)
            # (2,2,1): rows . pair(c,d)-slash . chi1(m)
            I.ldw("chm", lay.CHI + 8 * m)
            I.L("const W4<R> xp = slash_col(pcd, chm);"); I.flops += FL5["slash_col"]
            I.L("{ const Cx<R> " + ", ".join("a%d = row_col(%s, xp)" % (k, rn) for k, (rn, _) in enumerate(rows)) + ";"); I.flops += len(rows) * FL5["row_col"]
            for k, (rn, rcol) in enumerate(rows):
                I.jamp("a%d" % k, c_close(rcol, cpair(c, d), cchi(m)), pidx)
            I.flush_direct()
            I.L("}")
            I.L("}")
        insts.append(I)
    rows2_insts = insts
    if not cache_cols:
        add_group("rows2", rows2_insts, 1)
    # ---- cols2 loop: B = {c,d}; q1(x) . pair(P)-slash . chi2(B)
    insts = []
    for (c, d) in lay.PAIR:
        rest = rest_of(c, d)
        I = Inst5(lay, stride)
        I.leaf("ec", c); I.leaf("ed", d)
        I.ldw("pcd", lay.PAIR[(c, d)])
        cols = emit_cols2(I, c, d, "pcd", "ec", "ed")
        if cache_cols:      # parked for the three rows2 sub-blocks that need the same two currents (this loop then runs first)
            vec = I.P(2 * pair_index[(c, d)])
            I.L("sc_stw<R>(sc, %s, %s); sc_stw<R>(sc, %s + 1, %s);" % (vec, cols[0][0], vec, cols[1][0]))
        I.namp += 3 * (3 - len(cols))
        for x in rest:
            p = spair([l for l in rest if l != x])
            I.L("{")
            f0 = I.flops
            I.leaf("ex", x); I.qvec("qx", [x]); I.fv("ub")
            I.L("const W4<R> q1x = quark_step2(ub, ex, qx, mt, %s);" % I.iq(x)); I.flops += FL5["quark_step2"]
            I.redundant += I.flops - f0
            I.ldw("pp", lay.PAIR[p])
            I.L("const W4<R> r = row_slash(q1x, pp);"); I.flops += FL5["row_slash"]
            I.L("const Cx<R> " + ", ".join("a%d = row_col(r, %s)" % (k, cn) for k, (cn, _) in enumerate(cols)) + ";"); I.flops += len(cols) * FL5["row_col"]
            for k, (cn, ccol) in enumerate(cols):
                I.jamp("a%d" % k, c_close(cq1(x), cpair(*p), ccol), pidx)
            I.flush_direct()
            I.L("}")
        insts.append(I)
    add_group("cols2", insts, 1)
    if cache_cols:
        groups[-1][1].cache_vectors = 2 * len(lay.PAIR)
        add_group("rows2", rows2_insts, 1)
    return lay, groups


# ------------------------------------------------------------------------------------------
# kernel 3: four-gluon sub-trees built from pairs (V3(pair,pair), V4(pair,eps,eps)) closing three ways with the last
# gluon w, and the contact term V4(pair, pair, eps) on the bare line
# ------------------------------------------------------------------------------------------
def build_k3(stride, pidx, jacc=0, tm=()):
    # no Q1 / CHI slots: the one-gluon quark currents are needed exactly once each (in `ends`) and are formed there:
    # 214 slots per thread -> 128 threads per CTA
    lay = Layout5(want_pairs=True, want_iq_mid=False, jacc=jacc, want_q1chi=False, tm=tm)
    groups = []
    add_group = _grouper(groups)
    phase_a(lay, stride, add_group, want_pairs=True)
    def ends(I, w, quad):
        """the three four-vectors a quad term is dotted with: bilinears of the fermion ends and the dual of V3(quad, eps_w)"""
        I.leaf("ew", w); I.kvec("kw", [w]); I.kvec("kq", quad)
        f0 = I.flops
        I.qvec("qw", [w]); I.qvec("qq", quad)
        I.L("const W4<R> q1w = quark_step2(ub, ew, qw, mt, %s), chw = col_step(slash_col(ew, vv), qq, mt, %s);" % (I.iq(w), I.iq(*quad)))
        I.flops += FL5["quark_step2"] + FL5["slash_col"] + FL5["col_step"]
        I.redundant += I.flops - f0                    # kernel 2 forms the same ten currents
        I.L("const R ik4 = %s;" % I.ik2(*quad))
        # the last gluon w closes a sub-tree Q three ways: on the t~ end (colour Q.w), on the t end (w.Q), or through a three-gluon
        # vertex on the bare line, whose colour is the commutator Q.w - w.Q: its current x3 is folded into the other two,
        # which leaves two dot products and two jamp groups per sub-tree term instead of three
        I.L("const W4<R> x3 = v3_dual(ew, jtt, kq, kw, %s);" % I.ik2(*range(N)))
        I.L("const W4<R> x1 = wadd(bilinear(ub, chw), x3), x2 = wsub(bilinear(q1w, vv), x3);")
        I.flops += 2 * FL5["wadd"] + 2 * FL5["bilinear"] + FL5["v3_dual"]

    def close3(I, w, tname, col, k=""):
        """amplitudes of one four-gluon sub-tree term with the two ends (the V3 closing on the bare line is inside both); the caller flushes"""
        I.L("const Cx<R> a1%s = wdot(%s, x1), a2%s = wdot(%s, x2);" % (k, tname, k, tname)); I.flops += 2 * FL5["wdot"]
        I.namp += 1                 # the V3 closing is inside a1 and a2
        I.jamp("a1%s" % k, c_close(ONE, col, cchi(w)), pidx)
        I.jamp("a2%s" % k, c_close(cq1(w), col, ONE), pidx)

    # one instance per last gluon w: the three end vectors are formed once, then two nested table-driven loops run over the
    # 3 + 6 four-gluon sub-trees (unrolled they were ~8 k instructions and instruction-fetch bound; as 45 independent small
    # instances they rebuilt the end vectors 45 times: 38 % of this kernel's flops)
    insts = []
    for w in range(N):
        quad = rest_of(w)
        I = Inst5(lay, stride)
        ends(I, w, quad)
        a0 = quad[0]
        inners = []
        for b0 in quad[1:]:
            p1 = (a0, b0); p2 = spair([l for l in quad if l not in p1])
            J = Inst5(lay, stride, inner=True, parent=I if jacc else None)
            J.ldw("p1", lay.PAIR[p1]); J.ldw("p2", lay.PAIR[p2]); J.kvec("k1", list(p1)); J.kvec("k2", list(p2))
            J.L("const W4<R> t = v3_current(p1, p2, k1, k2, ik4);"); J.flops += FL5["v3_current"]
            close3(J, w, "t", c_v3(cpair(*p1), cpair(*p2)))
            J.flush_jamps() if jacc else J.flush_direct()
            inners.append(J)
        I.inner_loop("v3", inners)
        inners = []
        for p in [(quad[i], quad[j]) for i in range(4) for j in range(i + 1, 4)]:
            l1, l2 = [l for l in quad if l not in p]
            J = Inst5(lay, stride, inner=True, parent=I if jacc else None)
            J.ldw("pp", lay.PAIR[p]); J.leaf("e1", l1); J.leaf("e2", l2)
            J.L("const V4Dots<R> dots = v4_dots(pp, e1, e2, ik4);"); J.flops += FL5["v4_dots"]
            for k in range(3):          # the three contact structures share colour flows: their nine amplitudes are combined first
                J.L("const W4<R> t%d = v4_current(%d, dots, pp, e1, e2);" % (k, k)); J.flops += FL5["v4_current"]
                close3(J, w, "t%d" % k, c_v4(k, cpair(*p), c_leaf(l1), c_leaf(l2)), "_%d" % k)
            J.flush_jamps() if jacc else J.flush_direct()
            inners.append(J)
        I.inner_loop("v4", inners)
        if jacc:
            I.flush_global()
        insts.append(I)
    add_group("quads", insts, 1)
    # ---- V4(pair, pair', eps_m) on the bare line
    insts = []
    for m in range(N):
        quad = rest_of(m)
        a0 = quad[0]
        for b0 in quad[1:]:
            p1 = (a0, b0); p2 = spair([l for l in quad if l not in p1])
            I = Inst5(lay, stride)
            I.ldw("p1", lay.PAIR[p1]); I.ldw("p2", lay.PAIR[p2]); I.leaf("em", m)
            I.L("const V4Dots<R> dots = v4_dots(p1, p2, em, %s);" % I.ik2(*range(N))); I.flops += FL5["v4_dots"]
            for k in range(3):
                I.L("const Cx<R> b%d = wdot(v4_current(%d, dots, p1, p2, em), jtt);" % (k, k)); I.flops += FL5["v4_current"] + FL5["wdot"]
                I.jamp("b%d" % k, c_close(ONE, c_v4(k, cpair(*p1), cpair(*p2), c_leaf(m)), ONE), pidx)
            I.flush_direct()
            insts.append(I)
    add_group("pair_pair_v4", insts, 1)
    return lay, groups


# ------------------------------------------------------------------------------------------
# kernel 3, sharing form (include/me.h ME_OPT_SHARE_CURRENTS): the same diagrams as build_k3, organised
# around what depends on the gluon helicities only.  For the last gluon w the 21 four-gluon currents on quad = rest_of(w) (three
# V3(pair, pair'), eighteen V4(pair, eps, eps)) have colour factors in the six-dimensional space of multilinear Lie polynomials in the
# four generators; expanded on the left-normed brackets D_pi = [[[q0, q_pi1], q_pi2], q_pi3] they become six colour-ordered currents
#     U_pi = sum_T alpha_pi(T) V_T          (alpha_pi(T) = coefficient of the string q0 q_pi1 q_pi2 q_pi3 in the colour factor of T)
# that are formed ONCE for the (up to four) quark-helicity assignments a CTA loops over (pre-groups, run before the helicity loop), and
# each helicity costs twelve dot products U_pi . x1, U_pi . x2 with the two end vectors per last gluon.  Every colour flow of a
# (w, helicity) block is then complete in registers: the 48 flows go out by one RED pair each and no local jamp accumulators exist.
# The thirty currents stay on chip for the whole group (20 in tensor memory next to the pair currents, 10 in shared memory: one
# 128-thread CTA per SM in FP64, two in FP32 with one TMEM column per slot); the helicity loop stays outermost, so that all reductions
# into one staging row happen close in time (with the loop over w outside, the rows of four helicities per CTA no longer fit the L2
# and every reduction became a DRAM read-modify-write: 35 GB per launch instead of 9).
# ------------------------------------------------------------------------------------------
NU_SMEM = 2          # colour-ordered currents per last gluon kept in shared memory; the other four in tensor memory


def build_k3s(stride, pidx, cache_u=None):
    cache_u = K3S_CACHE_U if cache_u is None else cache_u
    if cache_u:
        # the thirty ordered currents of a group live in the L2-resident current cache (vector 6 w + k): what stays on chip (pair currents and
        # the 24 ordered contact amplitudes in tensor memory, 76 slots in shared memory) lets two CTAs share an SM
        lay = Layout5(want_pairs=True, want_iq_mid=False, jacc=24, want_q1chi=False, ik2_sizes=(2, 4, 5), tm=("PAIR", "J"))
    else:
        lay = Layout5(want_pairs=True, want_iq_mid=False, jacc=24, want_q1chi=False, ik2_sizes=(2, 4, 5), tm=("PAIR", "U"), nu=6, nu_smem=NU_SMEM)      # jacc: the 24 ordered contact amplitudes
    groups = []
    add_group = _grouper(groups)
    phase_a(lay, stride, add_group, want_pairs=True)          # the ten pair currents: gluon helicities only, once per group
    pis = list(permutations((1, 2, 3)))
    bases = {}
    insts = []
    for w in range(N):
        quad = rest_of(w)
        I = Inst5(lay, stride)
        # c_v3(x, y) = -[x, y]: three nested c_v3 give -[[[q0, a], b], c]; the coefficient of the string q0 a b c in it is -1
        basis = [c_v3(c_v3(c_v3(c_leaf(quad[0]), c_leaf(quad[q[0]])), c_leaf(quad[q[1]])), c_leaf(quad[q[2]])) for q in pis]
        bases[w] = basis
        I.L("W4<R> " + ", ".join("U%d" % k for k in range(6)) + ";")
        I.L("const R ik4 = %s;" % I.ik2(*quad))
        started = [False] * 6

        def accumulate(expr, X):
            alpha = [-X.get((quad[0], quad[q[0]], quad[q[1]], quad[q[2]]), 0) for q in pis]
            chk = {}
            for al, D in zip(alpha, basis):
                for st, v in D.items():
                    chk[st] = chk.get(st, 0) + al * v
            assert not _cdiff(X, chk, {}), "colour factor outside the span of the left-normed brackets"
            I.L("{ const W4<R> V = %s;" % expr)
            for k, al in enumerate(alpha):
                if al == 0:
                    continue
                assert al in (1, -1), al
                if not started[k]:
                    I.L("  U%d = %s;" % (k, "V" if al > 0 else "wsub(W4<R>{(R)0, (R)0, (R)0, (R)0, (R)0, (R)0, (R)0, (R)0}, V)"))
                    started[k] = True
                    I.flops += 0 if al > 0 else 8
                else:
                    I.L("  U%d = %s(U%d, V);" % (k, "wadd" if al > 0 else "wsub", k)); I.flops += 8
            I.L("}")

        a0 = quad[0]
        for b0 in quad[1:]:
            p1 = (a0, b0); p2 = spair([l for l in quad if l not in p1])
            I.L("{")
            I.ldw("p1", lay.PAIR[p1]); I.ldw("p2", lay.PAIR[p2]); I.kvec("k1", list(p1)); I.kvec("k2", list(p2))
            I.flops += FL5["v3_current"]
            accumulate("v3_current(p1, p2, k1, k2, ik4)", c_v3(cpair(*p1), cpair(*p2)))
            I.L("}")
        for p in [(quad[i], quad[j]) for i in range(4) for j in range(i + 1, 4)]:
            l1, l2 = [l for l in quad if l not in p]
            I.L("{")
            I.ldw("pp", lay.PAIR[p]); I.leaf("e1", l1); I.leaf("e2", l2)
            I.L("const V4Dots<R> dots = v4_dots(pp, e1, e2, ik4);"); I.flops += FL5["v4_dots"]
            for k in range(3):
                I.flops += FL5["v4_current"]
                accumulate("v4_current(%d, dots, pp, e1, e2)" % k, c_v4(k, cpair(*p), c_leaf(l1), c_leaf(l2)))
            I.L("}")
        assert all(started)
        if cache_u:
            I.L(" ".join("sc_stw<R>(sc, %s + %d, U%d);" % (I.P(6 * w), k, k) for k in range(6)))
        else:
            for k in range(6):
                I.stw(lay.U[(w, k)], "U%d" % k)
        insts.append(I)
    add_group("ubuild", insts, 1)
    for _, t, _, _ in groups:
        t.pre = True                                              # run once per group of helicities, before the helicity loop
        t.group_flops = t.flops; t.flops = 0
    if cache_u:
        groups[-1][1].cache_vectors = 6 * N
    # ---- per helicity: the two end vectors of w (bilinears of the fermion ends with the dual of V3(quad, eps_w) folded in) and 12 dots
    insts = []
    for w in range(N):
        quad = rest_of(w)
        I = Inst5(lay, stride)
        if cache_u:        # the first three ordered currents are requested before the end vectors are built, the other three before the first dots
            ubase = I.P(6 * w)
            I.L("const W4<R> " + ", ".join("u%d = sc_ldw<R>(sc, %s + %d)" % (k, ubase, k) for k in range(3)) + ";")
        I.leaf("ew", w); I.kvec("kw", [w]); I.kvec("kq", quad)
        f0 = I.flops
        I.qvec("qw", [w]); I.qvec("qq", quad)
        I.L("const W4<R> q1w = quark_step2(ub, ew, qw, mt, %s), chw = col_step(slash_col(ew, vv), qq, mt, %s);" % (I.iq(w), I.iq(*quad)))
        I.flops += FL5["quark_step2"] + FL5["slash_col"] + FL5["col_step"]
        I.redundant += I.flops - f0                    # kernel 2 forms the same ten one-gluon quark currents
        I.L("const W4<R> x3 = v3_dual(ew, jtt, kq, kw, %s);" % I.ik2(*range(N)))
        I.L("const W4<R> x1 = wadd(bilinear(ub, chw), x3), x2 = wsub(bilinear(q1w, vv), x3);")
        I.flops += 2 * FL5["bilinear"] + FL5["v3_dual"] + 2 * FL5["wadd"]
        if cache_u:
            I.L("const W4<R> " + ", ".join("u%d = sc_ldw<R>(sc, %s + %d)" % (k, ubase, k) for k in range(3, 6)) + ";")
        for k0 in (0, 3):                              # three currents in flight at a time
            if not cache_u:
                for k in range(k0, k0 + 3):
                    I.ldw("u%d" % k, lay.U[(w, k)])
            I.L("const Cx<R> " + ", ".join("a1_%d = wdot(u%d, x1), a2_%d = wdot(u%d, x2)" % (k, k, k, k) for k in range(k0, k0 + 3)) + ";")
        I.flops += 12 * FL5["wdot"]
        for k in range(6):
            I.jamp("a1_%d" % k, c_close(ONE, bases[w][k], cchi(w)), pidx)
            I.jamp("a2_%d" % k, c_close(cq1(w), bases[w][k], ONE), pidx)
        I.namp += 63 - 12                      # 21 four-gluon terms x three closings, carried by the twelve ordered amplitudes
        I.flush_direct()
        insts.append(I)
    add_group("quads", insts, 1)
    # ---- V4(pair, pair', eps_m) on the bare line.  Their 45 colour factors are multilinear Lie polynomials in the five generators: expanded
    # on the 24 left-normed brackets E_rho = [[[[0, r1], r2], r3], r4] (coefficient = coefficient of the string 0 r1 r2 r3 r4) the 45 amplitudes
    # add up to 24 ordered amplitudes Z_rho, accumulated in shared memory (table-driven slots), and every one of the 120 colour flows leaves
    # with ONE reduction pair as a combination of the Z_rho that contain it (360 pairs per helicity before: the reductions, not the arithmetic,
    # bound this kernel: 4.7 TB/s of reduction payload into the L2 in FP64 and FP32 alike)
    rhos = list(permutations((1, 2, 3, 4)))
    ebasis = [c_v3(c_v3(c_v3(c_v3(c_leaf(0), c_leaf(q[0])), c_leaf(q[1])), c_leaf(q[2])), c_leaf(q[3])) for q in rhos]
    assert all(E[(0,) + q] == 1 for E, q in zip(ebasis, rhos))
    for m_class in (True, False):               # m = gluon 0 (three instances) / m != 0 (twelve): two shapes of the update pattern
        insts = []
        for m in range(N):
            if (m == 0) != m_class:
                continue
            quad = rest_of(m)
            a0 = quad[0]
            for b0 in quad[1:]:
                p1 = (a0, b0); p2 = spair([l for l in quad if l not in p1])
                I = Inst5(lay, stride)
                I.ldw("p1", lay.PAIR[p1]); I.ldw("p2", lay.PAIR[p2]); I.leaf("em", m)
                I.L("const V4Dots<R> dots = v4_dots(p1, p2, em, %s);" % I.ik2(*range(N))); I.flops += FL5["v4_dots"]
                ups = []
                for k in range(3):
                    I.L("const Cx<R> b%d = wdot(v4_current(%d, dots, p1, p2, em), jtt);" % (k, k)); I.flops += FL5["v4_current"] + FL5["wdot"]
                    X = c_v4(k, cpair(*p1), cpair(*p2), c_leaf(m))
                    alpha = [X.get((0,) + q, 0) for q in rhos]
                    chk = {}
                    for al, E in zip(alpha, ebasis):
                        for st, v in E.items():
                            chk[st] = chk.get(st, 0) + al * v
                    assert not _cdiff(X, chk, {}) and all(al in (0, 1, -1) for al in alpha)
                    for sign in (1, -1):             # plus terms first: the same code for every instance of the class, the slots from the table
                        for r, al in enumerate(alpha):
                            if al == sign:
                                o = I.P(eo(lay.J + 2 * r, stride))
                                ups.append((o, "%sb%d.re" % ("" if sign > 0 else "-", k), "%sb%d.im" % ("" if sign > 0 else "-", k)))
                                I.flops += 2
                    I.namp += 1
                I.jamp_codes.extend(1 if u[1].startswith("-") else 0 for u in ups)     # (shape check of the looped instances)
                # an ordered amplitude may receive several of the three terms of one instance: its updates must not be split over batches that
                # read before an earlier one has written; batches of distinct slots only
                seen, batch = set(), []
                for u_ in ups:
                    slot = I.params[int(u_[0][3:-1])]
                    if slot in seen:
                        I.emit_accumulate(batch); seen, batch = set(), []
                    seen.add(slot); batch.append(u_)
                I.emit_accumulate(batch)
                insts.append(I)
        add_group("contact_m0" if m_class else "contact", insts, 1)
    I = Inst5(lay, stride)
    if I.in_tm(lay.J):
        I.L("xwait_st<TM>();")
    for r0 in range(0, 24, 4):
        if I.in_tm(lay.J):     # four ordered amplitudes per tcgen05.ld x16, cleared with one tcgen05.st x16
            o = eo(lay.J + 2 * r0, stride)
            I.L("XW<R, TM> zx%d; xldw_issue<R, TM>(zx%d, sm, tm, %d);" % (r0, r0, o))
            I.L("const W4<R> zw%d = xldw_get<R, TM>(zx%d);" % (r0, r0))
            I.L("xstw<R, TM>(sm, tm, %d, W4<R>{(R)0, (R)0, (R)0, (R)0, (R)0, (R)0, (R)0, (R)0});" % o)
            for k in range(4):
                I.L("const Cx<R> Z%d = {zw%d.r%d, zw%d.i%d};" % (r0 + k, r0, k, r0, k))
        else:
            for r in range(r0, r0 + 4):
                I.L("R zr%d, zi%d; cget<R>(sm + %d, zr%d, zi%d); cset<R>(sm + %d, (R)0, (R)0);" % (r, r, eo(lay.J + 2 * r, stride), r, r, eo(lay.J + 2 * r, stride)))
                I.L("const Cx<R> Z%d = {zr%d, zi%d};" % (r, r, r))
    for r in range(24):
        I.jamp("Z%d" % r, c_close(ONE, ebasis[r], ONE), pidx)
    I.namp -= 24
    I.flush_direct()
    add_group("contact_flush", [I], 1)
    return lay, groups


# ------------------------------------------------------------------------------------------
# source emission
# ------------------------------------------------------------------------------------------
def prologue_lines(lay):
    """per-event, helicity-independent: momenta -> signed gluon momenta, propagator denominators (FP64 from pairwise
    invariants, then rounded to R), polarisation bases, spinor bases"""
    sgn = lambda l: 1 if l < 2 else -1
    part = lambda l: l if l < 2 else l + 2
    out, fixed = [], 0
    A = out.append
    A("const double* pm = mom + (e >> 5) * (%d * 4 * 32) + (e & 31);" % NPAR)
    for k in range(NPAR):
        A("const P4<double> pd%d = {pm[%d], pm[%d], pm[%d], pm[%d]};" % (k, (4 * k) * 32, (4 * k + 1) * 32, (4 * k + 2) * 32, (4 * k + 3) * 32))
    lines, fl = dd_invariant_lines(range(N), range(N), sgn, part)      # exact invariants (hel_amp.cuh "Propagator denominators")
    out.extend(lines)
    fixed += fl
    for l in range(N):
        A("stp<R>(sm, %d, pcast<R>(%s));" % (lay.MOM + 4 * l, "pd%d" % part(l) if sgn(l) > 0 else "pneg(pd%d)" % part(l)))
    A("stp<R>(sm, %d, pcast<R>(pd2));" % lay.PT)
    for m, slot in lay.IK2.items():
        e, fl = dd_k2([i for i in range(N) if m >> i & 1], sgn)
        A("sm[ME_EO(%d)] = (R)(1.0 / dd_value(%s));" % (slot, e)); fixed += fl + 2
    for m, slot in lay.IQ.items():
        e, fl = dd_q2([i for i in range(N) if m >> i & 1], sgn)
        A("sm[ME_EO(%d)] = (R)(1.0 / dd_value(%s));" % (slot, e)); fixed += fl + 2
    for l in range(N):
        A("{ GluonBasis<R> gb = gluon_basis(pcast<R>(pd%d)); gb.bx *= (R)%d; gb.by *= (R)%d; stgb<R>(sm, %d, gb); }" % (part(l), -sgn(l), -sgn(l), lay.GBS[l]))
        fixed += 22
    A("sbt = spinor_basis(pcast<R>(pd2), mt);")
    A("sbtb = spinor_basis(pcast<R>(pd3), mt);")
    fixed += 40
    return out, fixed


def emit_kernel(name, ki, lay, groups, BLOCK, only=None, delegate=None, delegate_init=False):
    """only: None (FP64 instances with part of the slots in tensor memory or all in shared memory, FP32 in shared memory) or 'tm' (every
    instance in its tensor-memory layout; ki is then a tag like '2d'); delegate: tag of the tensor-memory variant this kernel's
    launcher hands every precision to unless ME_NO_TMEM=1"""
    src = []
    S = src.append

    def emit_groups(gs):
        for gname, tmpl, rows, unroll in gs:
            S("    // ---- %s: %d instances" % (gname, len(rows)))
            S("#pragma unroll %d" % unroll)
            S("    for (int it = 0; it < %d; ++it) {" % len(rows))
            S("      const int* tb = tab_%s_o%s_%s[it];" % (name, ki, gname))
            for l in tmpl.lines:
                if "@SUB:" in l:
                    sname = l.split("@SUB:")[1].split("@")[0]
                    l = l.replace("@SUB:%s@" % sname, "tab_%s_o%s_%s_%s" % (name, ki, gname, sname))
                S("      " + l)
            S("    }")

    namp = sum(t.namp * len(rows) for _, t, rows, _ in groups)
    S("// GENERATED by paper_2303_18244_b200/codegen (orbit-looped emitter, emit_orbit5.py) — do not edit.")
    S("// g g -> t t~ g g g, diagram kernel %s: %d amplitude terms in %d looped shapes; %d shared-memory slots per thread." % (ki, namp, len(groups), lay.nslots))
    tm0 = getattr(lay, "TM0", None)
    S("#define ME_SM_STRIDE %d" % BLOCK)
    if tm0 is not None:
        assert BLOCK in (128, 256)
        S("#define ME_TM_SLOT0 %d" % tm0)
    S("#include \"hel_amp.cuh\"")
    S("#include \"kernels.h\"")
    S("#include \"multi.h\"")
    S("#include <stdlib.h>")
    S("namespace me {")
    for gname, tmpl, rows, _ in groups:
        S("__constant__ int tab_%s_o%s_%s[%d][%d] = {" % (name, ki, gname, len(rows), len(tmpl.params)))
        for r in rows:
            S("  {%s}," % ", ".join(str(v) for v in r))
        S("};")
        for sname, srows in getattr(tmpl, "subtables", []):
            S("__constant__ int tab_%s_o%s_%s_%s[%d][%d] = {" % (name, ki, gname, sname, len(srows), len(srows[0])))
            for r in srows:
                S("  {%s}," % ", ".join(str(v) for v in r))
            S("};")
    S("template <typename R, typename RJ, bool TM>")
    minb = MIN_CTAS_F32.get(str(ki), 0)
    bounds = "%d" % BLOCK if not minb else "%d, sizeof(R) == 4 ? %d : 1" % (BLOCK, minb)
    S("__global__ void __launch_bounds__(%s) k_%s_o%s(const double* __restrict__ mom, long npad, const unsigned char* __restrict__ hels, int nh,"
      " double mt_d, RJ* __restrict__ gjbase, const int* __restrict__ helpe, long n, void* __restrict__ cache) {" % (bounds, name, ki))
    S("  extern __shared__ __align__(16) unsigned char smem_raw[];")
    S("  R* sm = reinterpret_cast<R*>(smem_raw) + 2 * threadIdx.x;")
    S("  const long e0 = (long)blockIdx.x * blockDim.x + threadIdx.x;")
    S("  if (!TM && e0 >= npad) return;")
    S("  const bool live = e0 < npad;                    // TMEM kernel: warps past the end stay for the CTA-wide alloc / dealloc and skip the helicity loop")
    S("  const long e = live ? e0 : npad - 1;")
    S("  uint32_t tm = 0, tm_base = 0;")
    if tm0 is not None:
        S("  if constexpr (TM) {")
        S("    constexpr uint32_t tm_cols = sizeof(R) == 8 ? %du : %du;      // FP32 slots take one column" % (lay.tm_cols, max(32, lay.tm_cols // 2)))
        S("    __shared__ uint32_t tm_slot;")
        S("    tm_base = tm_alloc(&tm_slot, tm_cols * %d);" % (BLOCK // 128))
        S("    tm = tm_base + ((uint32_t)(threadIdx.x & 96) << 16) + (threadIdx.x >> 7) * tm_cols;      // this warp's quarter of the 128 lanes (and half of the columns)")
        S("  }")
    ncache = max([getattr(t, "cache_vectors", 0) for _, t, _, _ in groups])
    if ncache:      # this CTA's region of the current cache: [vector][4 pairs of reals][thread]
        S("  R* const sc = reinterpret_cast<R*>(cache) + ((size_t)(blockIdx.y * gridDim.x + blockIdx.x) * (%d * 8 * ME_SM_STRIDE) + 2 * threadIdx.x);" % ncache)
    S("  const R mt = (R)mt_d;")
    S("  const unsigned npad32 = (unsigned)npad;   // a slice holds <= 65536 events: 240 rows x npad elements fit 32 bits (cheap RED addresses)")
    S("  SpinorBasis<R> sbt, sbtb;")
    S("  {")
    pro, fixed = prologue_lines(lay)
    for l in pro:
        S("    " + l)
    if lay.FERM is not None:
        if tm0 is not None and lay.FERM["sbt"] >= tm0:
            S("    xstsb<R, TM>(sm, tm, ME_EO(%d), sbt); xstsb<R, TM>(sm, tm, ME_EO(%d), sbtb);" % (lay.FERM["sbt"], lay.FERM["sbtb"]))
        else:
            S("    stsb<R>(sm, %d, sbt); stsb<R>(sm, %d, sbtb);" % (lay.FERM["sbt"], lay.FERM["sbtb"]))
    S("  }")
    S("#pragma unroll")
    if tm0 is not None and lay.jacc and lay.J >= tm0:
        S("  for (int s = 0; s < %d; ++s) xstw<R, TM>(sm, tm, ME_EO(%d) + s * 8 * ME_SM_STRIDE, W4<R>{(R)0, (R)0, (R)0, (R)0, (R)0, (R)0, (R)0, (R)0});" % (lay.jacc // 4, lay.J))
    else:
        S("  for (int s = 0; s < %d; ++s) sm[ME_EO(%d + s)] = 0;" % (2 * lay.jacc, lay.J))
    has_pre = any(getattr(t, "pre", False) for _, t, _, _ in groups)
    init_staging = any(getattr(t, "init_staging", False) for _, t, _, _ in groups)
    S("  const int hc_end = !live ? 0 : (int)(blockIdx.y + 1) * ME_HEL_PER_CTA < nh ? (int)(blockIdx.y + 1) * ME_HEL_PER_CTA : nh;")
    if has_pre:
        # sharing kernel: the helicities of this CTA share their gluon helicities (the host groups the list: include/me.h); what depends on
        # the gluons only is formed once, with the first valid helicity of the group, before the helicity loop
        S("  int h0 = 255;")
        S("  if (helpe != nullptr) h0 = helpe[e < n ? e : n - 1];")
        S("  else for (int hc = (int)blockIdx.y * ME_HEL_PER_CTA; hc < hc_end; ++hc) if (h0 == 255 && hels[hc] != 255) h0 = hels[hc];")
        S("  if (h0 != 255 && live) {")
        S("    const int h = h0;")
        emit_groups([g for g in groups if getattr(g[1], "pre", False)])
        S("  }")
    S("  for (int hc = (int)blockIdx.y * ME_HEL_PER_CTA; hc < hc_end; ++hc) {")
    S("    const int h = helpe != nullptr ? helpe[e < n ? e : n - 1] : hels[hc];")
    S("    RJ* gj = gjbase + (long)hc * %d * npad + e;" % (2 * 120))
    if init_staging:
        S("    if (h == 255) {                               // padding of a grouped helicity list: this kernel initialises the staging rows, these to zero")
        S("      for (int r = 0; r < %d; ++r) gj[(unsigned)r * npad32] = (RJ)0;" % (2 * 120))
        S("      continue;")
        S("    }")
        if True:
            S("#pragma unroll 8")
            S("    for (int r = 0; r < %d; ++r) gj[(unsigned)r * npad32] = (RJ)0;      // the rows of this helicity start at zero (no memset of the staging buffer)" % (2 * 120))
    else:
        S("    if (h == 255) continue;                       // padding of a grouped helicity list")
    if lay.FERM is not None:
        S("    {")
        if tm0 is not None and lay.FERM["sbt"] >= tm0:
            S("      xwait_st<TM>();")
            S("      const W4<R> ub = spinor_ubar(xldsb<R, TM>(sm, tm, ME_EO(%d)), lam_of<R>(h, %d));" % (lay.FERM["sbt"], NPAR - 1 - 2))
            S("      const W4<R> vv = spinor_v(xldsb<R, TM>(sm, tm, ME_EO(%d)), lam_of<R>(h, %d));" % (lay.FERM["sbtb"], NPAR - 1 - 3))
            S("      xstw<R, TM>(sm, tm, ME_EO(%d), ub); xstw<R, TM>(sm, tm, ME_EO(%d), vv); xstw<R, TM>(sm, tm, ME_EO(%d), bilinear(ub, vv)); xwait_st<TM>();"
              % (lay.FERM["ub"], lay.FERM["vv"], lay.FERM["jtt"]))
        else:
            S("      const W4<R> ub = spinor_ubar(ldsb<R>(sm, %d), lam_of<R>(h, %d));" % (lay.FERM["sbt"], NPAR - 1 - 2))
            S("      const W4<R> vv = spinor_v(ldsb<R>(sm, %d), lam_of<R>(h, %d));" % (lay.FERM["sbtb"], NPAR - 1 - 3))
            S("      stw<R>(sm, %d, ub); stw<R>(sm, %d, vv); stw<R>(sm, %d, bilinear(ub, vv));" % (lay.FERM["ub"], lay.FERM["vv"], lay.FERM["jtt"]))
        S("    }")
    else:
        S("    const W4<R> ub = spinor_ubar(sbt, lam_of<R>(h, %d));" % (NPAR - 1 - 2))
        S("    const W4<R> vv = spinor_v(sbtb, lam_of<R>(h, %d));" % (NPAR - 1 - 3))
        S("    const W4<R> jtt = bilinear(ub, vv);")
    emit_groups([g for g in groups if not getattr(g[1], "pre", False)])
    S("  }")
    if tm0 is not None:
        S("  if constexpr (TM) tm_free(tm_base, (sizeof(R) == 8 ? %du : %du) * %d);" % (lay.tm_cols, max(32, lay.tm_cols // 2), BLOCK // 128))
    S("}")
    if delegate is not None:
        S("extern const MultiKernel mk_%s_o%s;" % (name, delegate))
    S("static cudaError_t launch_o%s(int precision, const MultiArgs& a) {" % ki)
    S("  // few helicities per CTA: many short CTAs, so the last partial wave costs little")
    S("  const dim3 grid((unsigned)((a.npad + %d - 1) / %d), (unsigned)((a.nh + ME_HEL_PER_CTA - 1) / ME_HEL_PER_CTA));" % (BLOCK, BLOCK))
    NO_TMEM = "    static const bool no_tmem = getenv(\"ME_NO_TMEM\") != nullptr && getenv(\"ME_NO_TMEM\")[0] == '1';   // A/B timing: shared-memory-only kernels"
    def launch_line(inst, smem, cast):
        S("      cudaFuncSetAttribute(k_%s_o%s<%s>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)%s);" % (name, ki, inst, smem))
        S("      cudaFuncSetAttribute(k_%s_o%s<%s>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);" % (name, ki, inst))
        S("      k_%s_o%s<%s><<<grid, %d, %s, a.stream>>>(a.mom, a.npad, a.hels, a.nh, a.mt, (%s*)a.gj, a.hel_per_event, a.n, a.cache);" % (name, ki, inst, BLOCK, smem, cast))
    S("  const size_t smf = sizeof(float) * %d * %d, smd = sizeof(double) * %d * %d, smt = sizeof(double) * %d * %d;" % (lay.nslots, BLOCK, lay.nslots, BLOCK, tm0 or 0, BLOCK))
    S("  (void)smf; (void)smd; (void)smt;")
    if only == "tm":
        assert tm0 is not None
        S("  const size_t smtf = sizeof(float) * %d * %d;" % (tm0, BLOCK))
        S("  if (precision == 2) {")
        launch_line("float, float, true", "smtf", "float")
        S("  } else {")
        launch_line("double, double, true", "smt", "double")
        S("  }")
    elif only == "f32":          # this form of the kernel serves FP32 only (the FP64 form of the same step is another kernel)
        S("  if (precision != 2) return cudaErrorInvalidValue;")
        launch_line("float, float, false", "smf", "float")
    elif only == "f64tm":        # ... and this one FP64 amplitudes in the tensor-memory layout only (sharing kernels: never run with ME_NO_TMEM=1)
        assert tm0 is not None
        S("  if (precision == 2) return mk_%s_o%s.launch(precision, a);" % (name, delegate))
        launch_line("double, double, true", "smt", "double")
    else:
        if delegate is not None:
            S(NO_TMEM)
            S("  if (!no_tmem) return mk_%s_o%s.launch(precision, a);     // the variant with local accumulators in tensor memory" % (name, delegate))
        if tm0 is not None and delegate is None:
            S(NO_TMEM)
        S("  if (precision == 2) {")
        launch_line("float, float, false", "smf", "float")
        S("  } else {")
        if tm0 is not None:
            S("    if (!no_tmem) {         // FP64 amplitudes: tensor-memory kernel (two CTAs per SM)")
            launch_line("double, double, true", "smt", "double")
            S("      return cudaGetLastError();")
            S("    }")
        launch_line("double, double, false", "smd", "double")
        S("  }")
    S("  return cudaGetLastError();")
    S("}")
    # bit p of the mask: the kernel this entry launches for precision p zeroes its staging rows itself
    own = 7 if init_staging else 0
    if only == "f64tm":
        own = (own & 3) | (4 if delegate_init else 0)
    S("extern const MultiKernel mk_%s_o%s = {launch_o%s, %d};" % (name, ki, ki, own))
    S("}  // namespace me")
    flops = sum(t.flops * len(rows) for _, t, rows, _ in groups)
    redundant = sum(getattr(t, "redundant", 0) * len(rows) for _, t, rows, _ in groups)
    group_flops = sum(getattr(t, "group_flops", 0) * len(rows) for _, t, rows, _ in groups)
    return "\n".join(src) + "\n", dict(amplitudes=namp, flops=flops, redundant=redundant, group_flops=group_flops, fixed=fixed, slots=lay.nslots, tm_slot0=tm0, tm_cols=getattr(lay, "tm_cols", 0),
                                       shapes={g: len(r) for g, _, r, _ in groups}, cache_vectors=ncache,
                                       group_redundant=sum(getattr(t, "group_redundant", 0) * len(rows) for _, t, rows, _ in groups))


def emit_orbit5_process(name="gg_ttxggg"):
    perms = list(permutations(range(N)))
    pidx = {p: i for i, p in enumerate(perms)}
    color_num, color_denom = color_matrix(perms)
    ncol = len(perms)
    files, kinfo = {}, []
    builders = tuple((lambda st, px, i=i: build_k1(st, px, i, K1_PARTS, init_staging=K1_INIT_STAGING[0])) for i in range(K1_PARTS)) + ((lambda st, px: build_k2(st, px, cache_cols=False)), build_k3)
    for ki, b in enumerate(builders):
        lay, groups = b(BLOCK1, pidx)
        last = ki == len(builders) - 1
        src, info = emit_kernel(name, ki, lay, groups, BLOCK1, delegate="%dd" % ki if last else None)
        files["gen_%s_o%d.cu" % (name, ki)] = src
        kinfo.append(info)
        if last:      # variant of the last kernel with local jamp accumulators in tensor memory (see TM_K3); the plain one is its ME_NO_TMEM=1 fallback
            lay2, groups2 = build_k3(BLOCK1, pidx, jacc=K3D_JACC, tm=TM_K3)
            src2, info2 = emit_kernel(name, "%dd" % ki, lay2, groups2, BLOCK1, only="tm")
            files["gen_%s_o%dd.cu" % (name, ki)] = src2
            info["fp64_variant"] = dict(slots=lay2.nslots, tm_slot0=lay2.TM0, tm_cols=lay2.tm_cols, flops=info2["flops"], redundant=info2["redundant"])
    # sharing form of the last kernel (build_k3s): used when the helicity list is grouped by gluon helicities (ME_OPT_SHARE_CURRENTS)
    lay3, groups3 = build_k3s(BLOCK1, pidx)
    src3, info3 = emit_kernel(name, "2s", lay3, groups3, BLOCK1, only="tm")
    files["gen_%s_o2s.cu" % name] = src3
    assert info3["amplitudes"] == kinfo[-1]["amplitudes"], (info3["amplitudes"], kinfo[-1]["amplitudes"])
    # sharing form of the first kernel: the gluon-only currents of the three-gluon sub-trees once per group of helicities
    info0s = None
    if K1_PRE and K1_PARTS == 1:
        # FP64: with the two (u, w) halves as a nested loop (70 KB loop body instead of 93 KB: instruction fetch); FP32: without (measured
        # 41.6 ms per pass against 44.3 ms with the nested loop, whose table-driven accumulator offsets cost more than the fetch saves)
        lay0, groups0 = build_k1(BLOCK1, pidx, uw_loop=K1S_UW_LOOP, pre=True, cache_q=K1_CACHE_Q[0], init_staging=K1_INIT_STAGING[0])
        src0, info0s = emit_kernel(name, "0s", lay0, groups0, BLOCK1, only="f64tm" if K1S_UW_LOOP else None, delegate="0f" if K1S_UW_LOOP else None,
                                    delegate_init=K1_INIT_STAGING[1])
        files["gen_%s_o0s.cu" % name] = src0
        assert info0s["amplitudes"] == kinfo[0]["amplitudes"]
        if K1S_UW_LOOP:
            lay0f, groups0f = build_k1(BLOCK1, pidx, uw_loop=False, pre=True, cache_q=K1_CACHE_Q[1], init_staging=K1_INIT_STAGING[1])
            src0f, info0f = emit_kernel(name, "0f", lay0f, groups0f, BLOCK1, only="f32")
            files["gen_%s_o0f.cu" % name] = src0f
            info0s["cache_vectors"] = max(info0s["cache_vectors"], info0f["cache_vectors"])    # one region serves both forms
            info0s["fp32_form"] = dict(flops=info0f["flops"], redundant=info0f["redundant"], cache_vectors=info0f["cache_vectors"])
    # sharing-path form of the second kernel: column currents of a helicity through the current cache
    info1s = None
    if K2_CACHE_COLS and K1_PARTS == 1:
        lay1, groups1 = build_k2(BLOCK1, pidx, cache_cols=True)
        src1, info1s = emit_kernel(name, "1s", lay1, groups1, BLOCK1)
        files["gen_%s_o1s.cu" % name] = src1
        assert info1s["amplitudes"] == kinfo[1]["amplitudes"]
    namp = sum(k["amplitudes"] for k in kinfo)
    assert namp == 1890, namp
    # colour sum in its symmetric form (S§8(d)): per part  sum_r x_r (C_rr x_r + 2 sum_{c<r} C_rc x_c), as for the smaller
    # processes; the DMMA kernel executes 240 of the 450 8x4 tiles (64 flops per event each), the FP32 kernels the dense form twice
    cs_flops = 2 * ncol * (ncol + 1) + 4 * ncol
    cs_executed = 2 * 240 * 64 + 4 * ncol
    head = 2 * FL5["spinor"] + FL5["bilinear"]
    executed = sum(k["flops"] for k in kinfo) + len(kinfo) * head + cs_executed
    # algorithmic: every current once -> drop the tagged recomputation and the repeated phase A / spinors of kernels 2,3
    # the pairs, q1 and chi1 loops as they would run once (reference layout with all slots)
    ref_groups = []
    phase_a(Layout5(want_pairs=True, want_iq_mid=True, jacc=12), BLOCK1, _grouper(ref_groups), want_pairs=True)
    pa = {g: t.flops * len(rows) for g, t, rows, _ in ref_groups}
    # needed once: the 10 pairs (untagged as pxy of the first kernel; kernels 2 and 3 both run the pairs loop again), the 5 + 5
    # one-gluon quark currents (chi1: kernel 2's loop; q1: every use is a tagged rebuild, so one set is taken back out of the
    # redundant count), the spinors and their bilinear (once, not once per kernel)
    redundant = sum(k["redundant"] for k in kinfo) + (len(kinfo) - 1) * head + 2 * pa["pairs"] - pa["q1"]
    algo = executed - redundant - (cs_executed - cs_flops)
    fixed = sum(k["fixed"] for k in kinfo)
    src = []
    S = src.append
    S("// GENERATED by paper_2303_18244_b200/codegen (emit_orbit5.py) — do not edit.  g g -> t t~ g g g process table.")
    S("#include \"kernels.h\"")
    S("#include \"multi.h\"")
    S("#include <stdlib.h>")
    S("namespace me {")
    for ki in range(len(kinfo)):
        S("extern const MultiKernel mk_%s_o%d;" % (name, ki))
    S("extern const MultiKernel mk_%s_o2s;" % name)
    if info0s is not None:
        S("extern const MultiKernel mk_%s_o0s;" % name)
    if info1s is not None:
        S("extern const MultiKernel mk_%s_o1s;" % name)
    S("static const MultiKernel* const parts_%s[%d] = {%s};" % (name, len(kinfo), ", ".join("&mk_%s_o%d" % (name, ki) for ki in range(len(kinfo)))))
    sh_names = ["o%d" % ki for ki in range(len(kinfo) - 1)] + ["o2s"]
    if info0s is not None:
        sh_names[0] = "o0s"
    if info1s is not None:
        sh_names[1] = "o1s"
    S("static const MultiKernel* const parts_sh_%s[%d] = {%s};" % (name, len(kinfo), ", ".join("&mk_%s_%s" % (name, k) for k in sh_names)))
    # current sharing: the helicity list is ordered by gluon helicities, the four quark-helicity assignments of each adjacent (rank table);
    # flops per event with it on, over the full helicity set: kernel o2 per helicity -> per group of four + per helicity
    fmask = (1 << T_BIT) | (1 << TB_BIT)
    order = sorted(range(1 << NPAR), key=lambda h: (h & ~fmask, h & fmask))
    rank = [order.index(h) for h in range(1 << NPAR)]
    S("static const unsigned char gray_rank_%s[%d] = {%s};" % (name, 1 << NPAR, ", ".join(str(r) for r in rank)))
    k2 = kinfo[-1]
    a2 = k2["flops"] - k2["redundant"] - pa["pairs"]                   # algorithmic part of kernel o2 per helicity (the pairs are counted once, elsewhere)
    nhel, ngroups = 1 << NPAR, (1 << NPAR) // HEL_PER_CTA
    shared_event = nhel * (algo - a2) + ngroups * (info3["group_flops"] - pa["pairs"]) + nhel * (info3["flops"] - info3["redundant"]) + fixed
    executed_shared = executed - k2["flops"] + info3["flops"] + info3["group_flops"] / HEL_PER_CTA
    cache_vectors = info3["cache_vectors"]      # one region serves the sharing kernels one after the other
    if info0s is not None:     # kernel o0 per helicity -> per group of four + per helicity
        k0 = kinfo[0]
        shared_event += -nhel * (k0["flops"] - k0["redundant"]) + nhel * (info0s["flops"] - info0s["redundant"]) \
            + ngroups * (info0s["group_flops"] - info0s["group_redundant"])
        executed_shared += -k0["flops"] + info0s["flops"] + info0s["group_flops"] / HEL_PER_CTA
        cache_vectors = max(cache_vectors, info0s["cache_vectors"])
    if info1s is not None:     # same algorithm; the executed count loses the rebuilt column currents
        executed_shared += -kinfo[1]["flops"] + info1s["flops"]
        assert kinfo[1]["flops"] - kinfo[1]["redundant"] == info1s["flops"] - info1s["redundant"]
        cache_vectors = max(cache_vectors, info1s["cache_vectors"])
    S("static const double color_num_%s[%d] = {%s};" % (name, ncol * ncol, ", ".join(str(float(x)) for row in color_num for x in row)))
    S("static cudaError_t launch_%s(int precision, const LaunchArgs& a) {" % name)
    S("  static const bool no_tmem = getenv(\"ME_NO_TMEM\") != nullptr && getenv(\"ME_NO_TMEM\")[0] == '1';   // the sharing kernel exists in its tensor-memory form only")
    S("  if (a.share && !no_tmem) return launch_multi(precision, a, parts_sh_%s, %d, %d, color_num_%s, %d);" % (name, len(kinfo), ncol, name, cache_vectors))
    S("  return launch_multi(precision, a, parts_%s, %d, %d, color_num_%s, 0);" % (name, len(kinfo), ncol, name))
    S("}")
    S("// staging buffer of one helicity chunk; with current sharing also the current cache of kernel o0s behind it (%d vectors per thread)" % cache_vectors)
    S("static size_t scratch_%s(int precision, long npad, int share, int) {" % name)
    S("  const size_t staging = multi_scratch_bytes(precision, npad, %d);" % ncol)
    S("  return share ? (staging + 255) / 256 * 256 + multi_cache_bytes(precision, npad, %d) : staging;" % cache_vectors)
    S("}")
    S("extern const ProcTable tab_%s = {%d, %d, %d, %d, %d, %d, {%r, %r, %r}, {%r, %r, %r}, %r, color_num_%s, launch_%s, scratch_%s, true, gray_rank_%s, %r, %d, %r};"
      % (name, N, 1240, namp, ncol, color_denom, len(kinfo) + 1, float(algo), float(algo), float(algo),
         float(executed), float(executed), float(executed), float(fixed), name, name, name, name, float(shared_event), fmask, float(executed_shared)))
    S("}  // namespace me")
    files["gen_%s_table.cu" % name] = "\n".join(src) + "\n"
    info = dict(n=N, ndiagrams=1240, namp=namp, ncol=ncol, color_denom=color_denom, flops_per_helicity=algo,
                flops_executed_per_helicity=executed, fixed_flops=fixed, colour_flops=cs_flops, kernels=kinfo, block=BLOCK1,
                flops_shared_event=shared_event, flops_executed_per_helicity_shared=executed_shared, kernel_o2s=info3, kernel_o0s=info0s)
    return files, info
