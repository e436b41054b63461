"""Orbit-looped emitter for g g -> t t~ g g (BASELINE.json config 4, the headline workload).

Why (profiles/r1_ttxgg_fp64_blocked_v2.md): fully unrolled per-helicity code is ~40 k SASS instructions
(~640 KB); on B200 the kernel then stalls on instruction fetch for half of its cycles.  The 123 diagrams
fall into a handful of SHAPES that differ only by a relabelling of the four gluons, so each shape is
emitted ONCE as a loop over its instances; everything that depends on the labels (shared-memory offsets
of operands, helicity bits, colour-flow indices) comes from a small __constant__ table.  The loop body is
straight-line register code; the whole helicity body is a few thousand instructions and stays in the
instruction cache.

Evaluation scheme (same Feynman diagrams, same amplitudes — one complex number per diagram term, 159 in
total — as emit.py), organised to cut work:
  * two-sided quark line: row currents grown from the t end (0..2 gluons attached) meet column currents
    grown from the t~ end (0..1 gluons), so no current with three attached gluons is ever formed;
  * amplitudes that share their two fermion ends use the bilinear J = row gamma col once and a 4-vector
    dot per diagram; three-gluon vertices closing on the bare line use the dual current (hel_amp.cuh v3_dual).
Storage: per-event constants, persistent currents (6 gluon pairs, 4+4 one-gluon quark currents) and the 24
jamps in per-thread shared-memory slots [slot][thread] (north_star "jamp staging in shared memory").
"""
from itertools import permutations

from .emit import FLOPS, colour_sum_lines, dd_invariant_lines, dd_k2, dd_q2
from .topology import _pmul, _pcomm, _pscale, color_matrix

N = 4
NPAR = 6
PARK_SB = True             # tensor-memory kernels: spinor bases of t and t~ in shared memory instead of 20 registers held across the helicity walk
MIN_SEG_STEPS = 8          # helicity-segment split of small batches: steps of the helicity list per segment at least (every segment starts with a full evaluation)
STATIC_MAX_EVENTS = 8192   # me_compute_static: events one call takes (its current cache is a file-scope device array of 64 CTAs x 208 KB = 13 MiB)
NSCVEC_TRIPLES = 8  # current sharing: vectors parked per thread in the L2-resident scratch: two ordered currents per three-gluon sub-tree,
NSCVEC_QUAD_END = 14  # the six colour-ordered four-gluon currents that close on the bare quark line,
NSCVEC = 26         # and the two column-side combinations of each of the six rows2 instances
FL = dict(FLOPS, col_step=63, quark_step2=127, v3_dual=158)
# The amplitudes are formed in colour-ordered combinations throughout (each is still a sum of whole diagram terms): two-gluon quark currents
# with the pair current folded into the two stepwise ones; the V3 closing of the last gluon folded into the two quark-end closings
# (colour T.w - w.T); three-gluon sub-trees as two ordered currents (V4 pieces in their channels, Jacobi identity).
# partial unrolling lets the operand loads of the next instance overlap the arithmetic of the current one
UNROLL = dict(pairs=6, q1=4, chi1=4, triples=1, rows2=1, q1_pair_chi=12, pair_pair=3, pair_v4=6)      # FP64 (255 registers, 4 warps/SM)
UNROLL_SH = dict(pairs=1, q1=1, chi1=1)      # FP64 sharing kernel (as loops the FP32 kernel is 17 % slower: table loads in front of its cheaper arithmetic)
UNROLL32 = dict(pairs=6, q1=4, chi1=4, triples=1, rows2=2, q1_pair_chi=12, pair_pair=3, pair_v4=6)    # FP32 (8 warps/SM, registers to spare)


def lam_bit(label, npar=NPAR):
    p = label if label < 2 else label + 2
    return npar - 1 - p


# ---- current sharing across helicities (include/me.h ME_OPT_SHARE_CURRENTS, second half).
# The sharing kernel walks the helicities in a reflected Gray order whose fastest bits are the quark helicities, so that a current
# made of gluons only survives as many steps as possible.  Position p of the Gray code (0 = flips every other step) -> helicity bit.
T_BIT, TB_BIT = NPAR - 1 - 2, NPAR - 1 - 3
GRAY_BITS = [T_BIT, TB_BIT, lam_bit(3), lam_bit(2), lam_bit(1), lam_bit(0)]      # t, t~, g3, g2, g1, g0 (g0 slowest: parity pairing keeps the first half)


def gray_walk():
    """the 64 helicity indices in walk order"""
    out = []
    for i in range(1 << NPAR):
        g = i ^ (i >> 1)
        out.append(sum(((g >> pos) & 1) << hb for pos, hb in enumerate(GRAY_BITS)))
    return out


def walk_count(mask, walk=None):
    """steps of the walk (the first one included) on which a current that depends on the helicity bits `mask` is re-evaluated"""
    walk = walk or gray_walk()
    return 1 + sum(1 for a, b in zip(walk, walk[1:]) if (a ^ b) & mask)


def dep_mask(gluons=(), t=False, tb=False):
    m = 0
    for l in gluons:
        m |= 1 << lam_bit(l)
    return m | (1 << T_BIT if t else 0) | (1 << TB_BIT if tb else 0)


class SlotAlloc:
    """Slot allocator for the paired shared-memory layout (hel_amp.cuh): vectors start on even slots; the odd
    slot left behind by a 5-real basis (and any alignment gap) is handed out to scalars first."""

    def __init__(self):
        self.n, self.holes = 0, []

    def vec(self, size):
        if self.n & 1:
            self.holes.append(self.n); self.n += 1
        s = self.n
        self.n += size
        if size & 1:
            self.holes.append(self.n); self.n += 1
        return s

    def scalar(self):
        if self.holes:
            return self.holes.pop(0)
        s = self.n; self.n += 1
        return s


def eo(slot, stride):
    """element offset of a slot in the per-thread R array (ME_EO of hel_amp.cuh)"""
    return (slot >> 1) * 2 * stride + (slot & 1)


class Layout:
    npar = NPAR

    def __init__(self):
        # Slot order: what stays in shared memory in every precision first (momenta, bases, column currents, propagator
        # denominators: TM0 = 98 slots), then the categories the FP64 kernels keep in tensor memory (hel_amp.cuh "Tensor memory
        # as a per-thread scratchpad": 6 gluon-pair currents, 4 row currents, 24 jamps = 128 slots = 256 TMEM columns).  The FP32
        # kernel keeps all 226 slots in shared memory (two CTAs per SM fit as it is).
        A = SlotAlloc()
        self.MOM = A.vec(4 * N)            # signed gluon momenta (+p incoming, -p outgoing)
        self.PT = A.vec(4)                 # p_t
        self.GBS = [A.vec(5) for _ in range(N)]
        self.CHI = A.vec(8 * N)
        masks2 = [m for m in range(1, 1 << N) if bin(m).count("1") >= 2]
        self.IK2 = {m: A.scalar() for m in masks2}
        masksq = [m for m in range(1, (1 << N) - 1)]
        self.IQ = {m: A.scalar() for m in masksq}
        self.TM0 = A.vec(0)                # first TMEM slot (even)
        pairs = [(a, b) for a in range(N) for b in range(a + 1, N)]
        self.PAIR = {p: A.vec(8) for p in pairs}
        self.Q1 = A.vec(8 * N)
        self.J = A.vec(2 * 24)
        self.nslots = A.n + (A.n & 1)
        self.tm_cols = 2 * (self.nslots - self.TM0)
        assert self.tm_cols <= 256 and self.TM0 <= 113, (self.TM0, self.tm_cols)   # two CTAs per SM: 256 of 512 columns, 113 slots of smem each


def mask_of(*labels):
    m = 0
    for l in labels:
        m |= 1 << l
    return m


def sum_expr(terms):
    """' + a.re - b.im' -> 'a.re - b.im' (no leading zero: 0 + x is not an identity for x = -0)"""
    t = terms.strip()
    if t.startswith("+ "):
        return t[2:]
    if t.startswith("- "):
        return "-" + t[2:]
    return t


class Inst:
    """One instance of a block: records parameters; emits lines only when it is the template."""

    def __init__(self, lay, stride):
        self.lay, self.stride = lay, stride
        self.params, self.lines, self.flops, self.namp = [], [], 0, 0
        self.jamp_codes = []
        self.pending = []          # (sigma, code, amp) waiting for flush_jamps()
        self.zcount = 0
        self.tm0 = getattr(lay, "TM0", None)      # slots >= tm0 live in tensor memory in the FP64 kernels (None: no TMEM)
        self.inflight = []         # 4-vector loads issued, not yet converted (TMEM loads are asynchronous)
        self.cond = []             # (helicity-bit mask, flops) of the parts the sharing kernel re-evaluates only when one of those helicities changed
        self._cond_open = None

    tbname = "tb"          # name of the parameter-table row pointer in the emitted loop body

    def P(self, v):
        self.params.append(int(v))
        return "%s[%d]" % (self.tbname, len(self.params) - 1)

    def off(self, slot):                       # shared-memory element offset of a slot
        return self.P(eo(slot, self.stride))

    def in_tm(self, slot):
        return self.tm0 is not None and slot >= self.tm0

    def L(self, s):
        for name in self.inflight:            # one tcgen05.wait::ld covers every load issued before it
            self.lines.append("const W4<R> %s = xldw_get<R, TM>(%s_x);" % (name, name))
        self.inflight = []
        self.lines.append(s)

    # ---- current sharing: the code between begin_cond / end_cond depends on the helicity bits `mask` only; the sharing
    # instantiation (SH) skips it on the steps of the walk that leave them unchanged (the result it left behind is still valid)
    def begin_cond(self, mask):
        assert self._cond_open is None
        self._cond_open = (mask, self.flops)
        self.L("if (!SH || (chg & %s)) {" % self.P(mask))

    def end_cond(self, close=True):
        mask, f0 = self._cond_open
        self._cond_open = None
        self.cond.append((mask, self.flops - f0))
        if close:
            self.L("}")

    # ---- operand helpers
    def leaf(self, name, l):
        self.L("const W4<R> %s = gluon_pol_s<R>(sm + %s, lam_of<R>(h, %s));" % (name, self.off(self.lay.GBS[l]), self.P(lam_bit(l, self.lay.npar))))
        self.flops += FL["gluon_pol"]

    def kvec(self, name, labels):
        terms = ["ldp<R>(sm + %s)" % self.off(self.lay.MOM + 4 * l) for l in labels]
        expr = terms[0]
        for t in terms[1:]:
            expr = "padd(%s, %s)" % (expr, t)
            self.flops += 4
        self.L("const P4<R> %s = %s;" % (name, expr))

    def qvec(self, name, labels):
        expr = "ldp<R>(sm + %d)" % eo(self.lay.PT, self.stride)
        for l in labels:
            expr = "psub(%s, ldp<R>(sm + %s))" % (expr, self.off(self.lay.MOM + 4 * l))
            self.flops += 4
        self.L("const P4<R> %s = %s;" % (name, expr))

    def ldw(self, name, slot):
        if self.in_tm(slot):
            self.lines.append("XW<R, TM> %s_x; xldw_issue<R, TM>(%s_x, sm, tm, %s);" % (name, name, self.off(slot)))
            self.inflight.append(name)
        else:
            self.lines.append("const W4<R> %s = ldw<R>(sm + %s);" % (name, self.off(slot)))     # does not end the in-flight group

    def stw(self, slot, name):
        if self.in_tm(slot):
            self.L("xstw<R, TM>(sm, tm, %s, %s); xwait_st<TM>();" % (self.off(slot), name))     # later loops read it with tcgen05.ld
        else:
            self.L("stw<R>(sm + %s, %s);" % (self.off(slot), name))

    def ik2(self, *labels):
        return "sm[%s]" % self.off(self.lay.IK2[mask_of(*labels)])

    def iq(self, *labels):
        return "sm[%s]" % self.off(self.lay.IQ[mask_of(*labels)])

    def jamp(self, amp, col, perm_index):
        """queue J_sigma += c * amp for every string of the colour polynomial `col`"""
        self.namp += 1
        for st, c in col.items():
            if c == 0:
                continue
            code = {1: 0, -1: 1, 1j: 2, -1j: 3}[complex(c) if not isinstance(c, int) else c]
            self.jamp_codes.append(code)
            self.pending.append((perm_index[st], code, amp))

    # ---- jamp updates.  code: 0 -> +1, 1 -> -1, 2 -> +i, 3 -> -i
    _MUL = {(0, 0): 0, (0, 1): 1, (0, 2): 2, (0, 3): 3, (1, 0): 1, (1, 1): 0, (1, 2): 3, (1, 3): 2,
            (2, 0): 2, (2, 1): 3, (2, 2): 1, (2, 3): 0, (3, 0): 3, (3, 1): 2, (3, 2): 0, (3, 3): 1}
    _INV = {0: 0, 1: 1, 2: 3, 3: 2}

    def grouped_updates(self):
        """pending (sigma, code, amp) -> [(sigma, unit code u, name of combination z)] with J_sigma += u * z; every
        distinct combination z = sum_k c_k a_k (up to a unit factor) is formed ONCE in registers"""
        order, by = [], {}
        for sigma, code, amp in self.pending:
            if sigma not in by:
                by[sigma] = []; order.append(sigma)
            by[sigma].append((code, amp))
        self.pending = []
        combos, out = {}, []
        for sigma in order:
            L = by[sigma]
            u = L[0][0]
            key = tuple((self._MUL[(self._INV[u], c)], a) for c, a in L)
            if len(key) == 1:
                out.append((sigma, u, key[0][1]))
                continue
            if key not in combos:
                name = "z%d_%d" % (self.zcount, len(combos))
                re = "".join({0: " + %s.re", 1: " - %s.re", 2: " - %s.im", 3: " + %s.im"}[c] % a for c, a in key)
                im = "".join({0: " + %s.im", 1: " - %s.im", 2: " + %s.re", 3: " - %s.re"}[c] % a for c, a in key)
                self.L("const Cx<R> %s = {%s, %s};" % (name, sum_expr(re), sum_expr(im)))
                self.flops += 2 * (len(key) - 1)
                combos[key] = name
            out.append((sigma, u, combos[key]))
        self.zcount += 1
        return out

    @staticmethod
    def unit_times(u, z):
        """(re, im) expressions of u * z"""
        return {0: ("%s.re" % z, "%s.im" % z), 1: ("-%s.re" % z, "-%s.im" % z),
                2: ("-%s.im" % z, "%s.re" % z), 3: ("%s.im" % z, "-%s.re" % z)}[u]

    JBATCH = 4     # accumulators read, updated and written back together (shared memory)
    JBATCH_TM = 8  # the same in tensor memory: more tcgen05.ld in flight per wait (FP64 -1 %; 8 in shared memory costs FP32 +1 %)

    def emit_accumulate(self, ups):
        """ups = [(shared-memory offset expression, re, im)]: J[offset] += (re, im).  The offsets are run-time values in the
        looped shapes, so the compiler must assume that consecutive read-modify-writes alias and chains them (load -> add ->
        store -> next load: one shared-memory latency per update, with one warp per scheduler to hide it).  The flows of one
        flush are distinct by construction: all loads of a batch are issued first, then the adds, then the stores."""
        if self.in_tm(self.lay.J):
            # jamps in tensor memory: tcgen05.ld x4 / st x4 per flow; the stores of the previous batch must have completed first
            def emit(jb):
                for b0 in range(0, len(ups), jb):
                    batch = ups[b0:b0 + jb]
                    # (the flows of one flush are distinct: only its first batch can read what an earlier flush stored)
                    self.L("{ R " + ", ".join("jr%d, ji%d" % (i, i) for i in range(len(batch))) + "; XC<R, TM> "
                           + ", ".join("jx%d" % i for i in range(len(batch))) + ";" + (" xwait_st<TM>();" if b0 == 0 else ""))
                    for i, (o, re, im) in enumerate(batch):
                        self.L("  xcget_issue<R, TM>(jx%d, sm, tm, %s);" % (i, o))
                    for i, (o, re, im) in enumerate(batch):
                        self.L("  xcget_get<R, TM>(jx%d, jr%d, ji%d);" % (i, i, i))
                    for i, (o, re, im) in enumerate(batch):
                        self.L("  xcset<R, TM>(sm, tm, %s, jr%d + (%s), ji%d + (%s));" % (o, i, re, i, im))
                    self.L("}")
            if len(ups) > self.JBATCH:          # batch size by instantiation: the shared-memory instance of the same template keeps 4
                self.L("if constexpr (TM) {"); emit(self.JBATCH_TM); self.L("} else {"); emit(self.JBATCH); self.L("}")
            else:
                emit(self.JBATCH)
            return
        for b0 in range(0, len(ups), self.JBATCH):
            batch = ups[b0:b0 + self.JBATCH]
            if len(batch) == 1:
                self.L("cacc<R>(sm + %s, %s, %s);" % batch[0])
                continue
            self.L("{ R " + ", ".join("jr%d, ji%d" % (i, i) for i in range(len(batch))) + ";")
            for i, (o, re, im) in enumerate(batch):
                self.L("  cget<R>(sm + %s, jr%d, ji%d);" % (o, i, i))
            for i, (o, re, im) in enumerate(batch):
                self.L("  cset<R>(sm + %s, jr%d + (%s), ji%d + (%s));" % (o, i, re, i, im))
            self.L("}")

    def flush_jamps(self):
        """one shared-memory read-modify-write (a single 128-bit load and store) per colour flow touched since the
        last flush; amplitudes that feed the same flow are combined in registers first"""
        ups = []
        for sigma, u, z in self.grouped_updates():
            re, im = self.unit_times(u, z)
            ups.append((self.off(self.lay.J + 2 * sigma), re, im))
            self.flops += 2
        self.emit_accumulate(ups)


# colour polynomials (phases folded in, see topology.py): strings are tuples of gluon labels
def c_leaf(l):
    return {(l,): 1}


def c_v3(x1, x2):
    return _pscale(_pcomm(x1, x2), -1)


def c_v4(k, x1, x2, x3):
    if k == 0:
        return _pcomm(_pcomm(x1, x2), x3)
    if k == 1:
        return _pcomm(_pcomm(x1, x3), x2)
    return _pscale(_pcomm(x1, _pcomm(x2, x3)), -1)


def c_step(prev, g):          # quark step (either end): phase i*i = -1
    return _pscale(_pmul(prev, g), -1)


def c_close(left, mid, right):  # closing vertex: phase i
    return _pscale(_pmul(_pmul(left, mid), right), 1j)


ONE = {(): 1}


def _cdiff(A, B, C):
    """colour polynomial A - (B - C); empty when the colour-ordering identity A = B - C holds"""
    out = dict(A)
    for P, k in ((B, -1), (C, 1)):
        for st, v in P.items():
            out[st] = out.get(st, 0) + k * v
    return {st: v for st, v in out.items() if abs(v) > 1e-12}


def build_groups(stride):
    lay = Layout()
    perms = list(permutations(range(N)))
    pidx = {p: i for i, p in enumerate(perms)}
    groups = []      # (name, template Inst, [param rows])

    def add_group(name, instances, mode="both"):
        """mode: 'both' | 'plain' (kernel instantiations without current sharing) | 'sh' (sharing instantiations only)"""
        tmpl = instances[0]
        tmpl.mode = mode
        for it in instances[1:]:
            assert it.lines == tmpl.lines, "instances of %s differ in shape" % name
            assert it.jamp_codes == tmpl.jamp_codes, "instances of %s differ in colour coefficients" % name
        tmpl.cond_all = [it.cond for it in instances]
        groups.append((name, tmpl, [it.params for it in instances]))

    labels = list(range(N))
    cpair = lambda a, b: c_v3(c_leaf(a), c_leaf(b))       # colour of the stored pair(a,b), a<b
    cq1 = lambda l: c_step(ONE, c_leaf(l))
    cchi = lambda l: c_step(c_leaf(l), ONE)

    # ---- A1: gluon pairs  V3(eps_a, eps_b)
    insts = []
    for (a, b) in lay.PAIR:
        I = Inst(lay, stride)
        I.begin_cond(dep_mask([a, b]))
        I.leaf("ea", a); I.leaf("eb", b)
        I.kvec("ka", [a]); I.kvec("kb", [b])
        I.L("const W4<R> t = v3_current(ea, eb, ka, kb, %s);" % I.ik2(a, b)); I.flops += FL["v3_current"]
        I.stw(lay.PAIR[(a, b)], "t")
        I.end_cond()
        insts.append(I)
    add_group("pairs", insts)
    # ---- A2: one-gluon row currents from the t end
    insts = []
    for l in labels:
        I = Inst(lay, stride)
        I.begin_cond(dep_mask([l], t=True))
        I.leaf("el", l); I.qvec("q", [l])
        I.L("const W4<R> t = quark_step2(ub, el, q, mt, %s);" % I.iq(l)); I.flops += FL["quark_step2"]
        I.stw(lay.Q1 + 8 * l, "t")
        I.end_cond()
        insts.append(I)
    add_group("q1", insts)
    # ---- A3: one-gluon column currents from the t~ end: chi_w = (qslash+m)/(q^2-m^2) eps_w-slash v, q = p_t - K_{all but w}
    insts = []
    for w in labels:
        rest = [l for l in labels if l != w]
        I = Inst(lay, stride)
        I.begin_cond(dep_mask([w], tb=True))
        I.leaf("ew", w); I.qvec("q", rest)
        I.L("const W4<R> t = col_step(slash_col(ew, vv), q, mt, %s);" % I.iq(*rest)); I.flops += FL["slash_col"] + FL["col_step"]
        I.stw(lay.CHI + 8 * w, "t")
        I.end_cond()
        insts.append(I)
    add_group("chi1", insts)
    # ---- B1: three-gluon sub-trees on {a,b,c} closing three ways with the remaining gluon w
    insts = []
    for vi, w in enumerate(labels):
        a, b, c = [l for l in labels if l != w]
        I = Inst(lay, stride)
        # colour-ordered form of the three-gluon sub-tree: the four-gluon-vertex pieces carry the colours of the three channels,
        # and the Jacobi identity col1 = col0 + col2 leaves two independent currents s0, s2 instead of six terms.  They depend
        # on the helicities of a, b, c only: the sharing kernel parks them in its L2-resident scratch (vectors 2 vi, 2 vi + 1)
        cols = [c_v3(cpair(a, b), c_leaf(c)), c_v3(cpair(a, c), c_leaf(b)), c_v3(cpair(b, c), c_leaf(a))] + \
               [c_v4(k, c_leaf(a), c_leaf(b), c_leaf(c)) for k in range(3)]
        assert all(not _cdiff(cols[3 + k], cols[k], {}) for k in range(3)) and not _cdiff(cols[1], cols[0], _pscale(cols[2], -1))
        I.L("W4<R> s0, s2;")
        I.begin_cond(dep_mask([a, b, c]))
        I.leaf("ea", a); I.leaf("eb", b); I.leaf("ec", c)
        I.kvec("ka", [a]); I.kvec("kb", [b]); I.kvec("kc", [c])
        I.L("const P4<R> kab = padd(ka, kb), kac = padd(ka, kc), kbc = padd(kb, kc);"); I.flops += 12
        I.ldw("pab", lay.PAIR[(a, b)]); I.ldw("pac", lay.PAIR[(a, c)]); I.ldw("pbc", lay.PAIR[(b, c)])
        I.L("const R ik3 = %s;" % I.ik2(a, b, c))
        I.L("const V4Dots<R> dots = v4_dots(ea, eb, ec, ik3);"); I.flops += FL["v4_dots"]
        I.L("const W4<R> t14 = wadd(v3_current(pac, eb, kac, kb, ik3), v4_current(1, dots, ea, eb, ec));")
        I.L("s0 = wadd(wadd(v3_current(pab, ec, kab, kc, ik3), v4_current(0, dots, ea, eb, ec)), t14);")
        I.L("s2 = wadd(wadd(v3_current(pbc, ea, kbc, ka, ik3), v4_current(2, dots, ea, eb, ec)), t14);")
        I.flops += 3 * (FL["v3_current"] + FL["v4_current"]) + 5 * 8
        I.namp += 4 * 3                              # diagram terms folded into the two ordered currents
        vec = I.P(2 * vi)
        I.L("if constexpr (SH) { sc_stw<R>(sc, %s, s0); sc_stw<R>(sc, %s + 1, s2); }" % (vec, vec))
        I.end_cond(close=False)
        I.L("} else {")
        I.L("  s0 = sc_ldw<R>(sc, %s); s2 = sc_ldw<R>(sc, %s + 1);" % (vec, vec))
        I.L("}")
        # the last gluon w closes the sub-tree three ways: on the t~ end (colour T.w), on the t end (w.T), or through a
        # three-gluon vertex on the bare line, whose colour is the commutator T.w - w.T: its dual current dd is folded into the
        # other two, which leaves two dot products and two jamp groups per ordered current
        I.leaf("ew", w); I.kvec("kabc", [a, b, c]); I.kvec("kw", [w])
        I.ldw("chiw", lay.CHI + 8 * w); I.ldw("q1w", lay.Q1 + 8 * w)
        I.L("const W4<R> dd = v3_dual(ew, jtt, kabc, kw, %s);" % I.ik2(a, b, c, w)); I.flops += FL["v3_dual"]
        I.L("const W4<R> j1 = wadd(bilinear(ub, chiw), dd), j2 = wsub(bilinear(q1w, vv), dd);"); I.flops += 2 * FL["bilinear"] + 16
        for nm, col in (("s0", cols[0]), ("s2", cols[2])):
            I.L("{")
            I.L("  const Cx<R> a1 = wdot(%s, j1), a2 = wdot(%s, j2);" % (nm, nm)); I.flops += 2 * FL["wdot"]
            I.namp += 1                                                   # V3(t, eps_w) on the bare line is inside a1 and a2
            I.jamp("a1", c_close(ONE, col, cchi(w)), pidx)                    # ubar . t-slash . chi_w
            I.jamp("a2", c_close(cq1(w), col, ONE), pidx)                     # q1(w) . t-slash . v
            I.flush_jamps()
            I.L("}")
        insts.append(I)
    add_group("triples", insts)
    # ---- B2: the three row currents with gluons {a,b} attached, each closing three ways on {c,d}
    insts = []
    for ri, (a, b) in enumerate(lay.PAIR):
        c, d = [l for l in labels if l not in (a, b)]
        I = Inst(lay, stride)
        # the two column-side combinations depend on the t~ helicity and the gluons c, d only: the sharing kernel parks them in its scratch
        I.L("W4<R> xcd, xdc;")
        I.begin_cond(dep_mask([c, d], tb=True))
        I.leaf("ec", c); I.leaf("ed", d)
        I.ldw("pcd", lay.PAIR[(c, d)])
        I.ldw("chic", lay.CHI + 8 * c); I.ldw("chid", lay.CHI + 8 * d)
        I.L("const W4<R> xp = slash_col(pcd, vv);"); I.flops += FL["slash_col"]
        I.L("xcd = wadd(slash_col(ec, chid), xp); xdc = wsub(slash_col(ed, chic), xp);"); I.flops += 2 * (FL["slash_col"] + 8)
        vec = I.P(NSCVEC_QUAD_END + 2 * ri)
        I.L("if constexpr (SH) { sc_stw<R>(sc, %s, xcd); sc_stw<R>(sc, %s + 1, xdc); }" % (vec, vec))
        I.end_cond(close=False)
        I.L("} else {")
        I.L("  xcd = sc_ldw<R>(sc, %s); xdc = sc_ldw<R>(sc, %s + 1);" % (vec, vec))
        I.L("}")
        I.leaf("ea", a); I.leaf("eb", b)
        I.ldw("pab", lay.PAIR[(a, b)])
        I.ldw("q1a", lay.Q1 + 8 * a); I.ldw("q1b", lay.Q1 + 8 * b)
        I.qvec("q", [a, b])
        I.L("const R iq2 = %s;" % I.iq(a, b))
        # colour-ordered two-gluon currents: the pair current (a commutator, colour ab - ba) is folded into the two stepwise
        # currents, on the row side before the common propagator and on the column side before the dot product; the nine
        # diagram terms of this block become four colour-ordered amplitudes, one colour flow each
        col_ab, col_ba = c_step(cq1(a), c_leaf(b)), c_step(cq1(b), c_leaf(a))
        assert not _cdiff(c_step(ONE, cpair(a, b)), col_ab, col_ba)
        for col in (col_ab, col_ba):
            assert not _cdiff(c_close(col, cpair(c, d), ONE), c_close(col, c_leaf(c), cchi(d)), c_close(col, c_leaf(d), cchi(c)))
        I.L("const W4<R> sp = row_slash(ub, pab);"); I.flops += FL["row_slash"]
        I.L("const W4<R> rab = row_step(wadd(row_slash(q1a, eb), sp), q, mt, iq2), rba = row_step(wsub(row_slash(q1b, ea), sp), q, mt, iq2);")
        I.flops += 2 * (FL["row_slash"] + 8 + FL["col_step"])
        I.L("const Cx<R> a1 = row_col(rab, xcd), a2 = row_col(rab, xdc), a3 = row_col(rba, xcd), a4 = row_col(rba, xdc);"); I.flops += 4 * FL["row_col"]
        I.jamp("a1", c_close(col_ab, c_leaf(c), cchi(d)), pidx)
        I.jamp("a2", c_close(col_ab, c_leaf(d), cchi(c)), pidx)
        I.jamp("a3", c_close(col_ba, c_leaf(c), cchi(d)), pidx)
        I.jamp("a4", c_close(col_ba, c_leaf(d), cchi(c)), pidx)
        I.namp += 5
        I.flush_jamps()
        insts.append(I)
    add_group("rows2", insts)
    # ---- B3: q1(x) . pair(y,z)-slash . chi_w
    insts = []
    for x in labels:
        for w in labels:
            if w == x:
                continue
            y, z = [l for l in labels if l not in (x, w)]
            I = Inst(lay, stride)
            I.ldw("q1x", lay.Q1 + 8 * x); I.ldw("pyz", lay.PAIR[(y, z)]); I.ldw("chiw", lay.CHI + 8 * w)
            I.L("const Cx<R> a1 = row_col(row_slash(q1x, pyz), chiw);"); I.flops += FL["row_slash"] + FL["row_col"]
            I.jamp("a1", c_close(cq1(x), cpair(y, z), cchi(w)), pidx)
            I.flush_jamps()
            insts.append(I)
    add_group("q1_pair_chi", insts)
    # ---- B4: V3(pair, pair') on the bare line
    insts = []
    for (a, b), (c, d) in (((0, 1), (2, 3)), ((0, 2), (1, 3)), ((0, 3), (1, 2))):
        I = Inst(lay, stride)
        I.ldw("pab", lay.PAIR[(a, b)]); I.ldw("pcd", lay.PAIR[(c, d)])
        I.kvec("kab", [a, b]); I.kvec("kcd", [c, d])
        I.L("const Cx<R> a1 = wdot(v3_current(pab, pcd, kab, kcd, %s), jtt);" % I.ik2(a, b, c, d)); I.flops += FL["v3_current"] + FL["wdot"]
        I.jamp("a1", c_close(ONE, c_v3(cpair(a, b), cpair(c, d)), ONE), pidx)
        I.flush_jamps()
        insts.append(I)
    add_group("pair_pair", insts, mode="plain")
    # ---- B5: four-gluon vertex (pair, eps_c, eps_d) on the bare line, three colour structures
    insts = []
    for (a, b) in lay.PAIR:
        c, d = [l for l in labels if l not in (a, b)]
        I = Inst(lay, stride)
        I.ldw("pab", lay.PAIR[(a, b)]); I.leaf("ec", c); I.leaf("ed", d)
        I.L("const V4Dots<R> dots = v4_dots(pab, ec, ed, %s);" % I.ik2(a, b, c, d)); I.flops += FL["v4_dots"]
        for k in range(3):
            I.L("const Cx<R> b%d = wdot(v4_current(%d, dots, pab, ec, ed), jtt);" % (k, k)); I.flops += FL["v4_current"] + FL["wdot"]
            I.jamp("b%d" % k, c_close(ONE, c_v4(k, cpair(a, b), c_leaf(c), c_leaf(d)), ONE), pidx)
        I.flush_jamps()
        insts.append(I)
    add_group("pair_v4", insts, mode="plain")
    # ---- B4 + B5 of the sharing kernel: the 21 four-gluon currents that close on the bare line (V3(pair, pair'), V4(pair, eps, eps)) depend
    # on the gluon helicities only, and their colour factors are multilinear Lie polynomials in the four generators, a six-dimensional
    # space with basis D_pi = [[[T0, T_pi1], T_pi2], T_pi3] (the coefficient of D_pi is the coefficient of the string 0 pi1 pi2 pi3).  So
    #     sum_T c_T (V_T . jtt) = sum_pi D_pi (U_pi . jtt),   U_pi = sum_T alpha_pi(T) V_T :
    # six colour-ordered currents per gluon-helicity assignment (re-evaluated 16 times per event, parked in the L2-resident scratch)
    # and six dot products with ubar gamma v per helicity
    I = Inst(lay, stride)
    pis = list(permutations((1, 2, 3)))
    basis = [_pcomm(_pcomm(_pcomm(c_leaf(0), c_leaf(q[0])), c_leaf(q[1])), c_leaf(q[2])) for q in pis]
    terms = []            # (emit function -> expression of V_T, colour polynomial X_T)
    I.begin_cond(dep_mask([0, 1, 2, 3]))
    I.L("W4<R> " + ", ".join("U%d" % k for k in range(6)) + ";")
    started = [False] * 6

    def accumulate(expr, X):
        alpha = [X.get((0,) + q, 0) for q in pis]
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

    ik4 = I.ik2(0, 1, 2, 3)
    I.L("const R ik4 = %s;" % ik4)
    for (a, b), (c, d) in (((0, 1), (2, 3)), ((0, 2), (1, 3)), ((0, 3), (1, 2))):
        I.L("{")
        I.ldw("pab", lay.PAIR[(a, b)]); I.ldw("pcd", lay.PAIR[(c, d)])
        I.kvec("kab", [a, b]); I.kvec("kcd", [c, d])
        I.flops += FL["v3_current"]
        accumulate("v3_current(pab, pcd, kab, kcd, ik4)", c_v3(cpair(a, b), cpair(c, d)))
        I.namp += 1
        I.L("}")
    for (a, b) in lay.PAIR:
        c, d = [l for l in labels if l not in (a, b)]
        I.L("{")
        I.ldw("pab", lay.PAIR[(a, b)]); I.leaf("ec", c); I.leaf("ed", d)
        I.L("const V4Dots<R> dots = v4_dots(pab, ec, ed, ik4);"); I.flops += FL["v4_dots"]
        for k in range(3):
            I.flops += FL["v4_current"]
            accumulate("v4_current(%d, dots, pab, ec, ed)" % k, c_v4(k, cpair(a, b), c_leaf(c), c_leaf(d)))
            I.namp += 1
        I.L("}")
    assert all(started)
    for k in range(6):
        I.L("sc_stw<R>(sc, %d, U%d);" % (NSCVEC_TRIPLES + k, k))
    I.end_cond()
    for k in range(6):
        I.L("const W4<R> u%d = sc_ldw<R>(sc, %d);" % (k, NSCVEC_TRIPLES + k))
    I.L("const Cx<R> " + ", ".join("q%d = wdot(u%d, jtt)" % (k, k) for k in range(6)) + ";"); I.flops += 6 * FL["wdot"]
    for k in range(6):
        I.jamp("q%d" % k, c_close(ONE, basis[k], ONE), pidx)
    I.namp -= 6                       # the six ordered amplitudes are sums of the 21 diagram terms counted above
    I.flush_jamps()
    add_group("quad_bare", [I], mode="sh")
    return lay, perms, groups


def emit_orbit_process(name="gg_ttxgg", block=128):
    stride = block
    lay, perms, groups = build_groups(stride)
    color_num, color_denom = color_matrix(perms)
    ncol = len(perms)
    cs_lines, cs_flops = colour_sum_lines(color_num, ncol, color_denom)
    namp = sum(t.namp * len(rows) for _, t, rows in groups if t.mode != "sh")
    assert namp == sum(t.namp * len(rows) for _, t, rows in groups if t.mode != "plain")       # both instantiations cover the same diagram terms
    flops = sum(t.flops * len(rows) for _, t, rows in groups if t.mode != "sh")
    per_hel = flops + cs_flops + 2 * FL["spinor"] + FL["bilinear"]
    sgn = lambda l: 1 if l < 2 else -1
    part = lambda l: l if l < 2 else l + 2
    src = []
    S = src.append
    S("// GENERATED by paper_2303_18244_b200/codegen (orbit-looped emitter) — do not edit.")
    S("// g g -> t t~ g g: 123 diagrams, %d amplitudes in %d looped shapes, 24 colour flows; %d shared-memory slots per thread." % (namp, len(groups), lay.nslots))
    S("#define ME_SM_STRIDE %d" % block)
    S("#define ME_TM_SLOT0 %d" % lay.TM0)
    S("#include \"hel_amp.cuh\"")
    S("#include \"kernels.h\"")
    S("#include <stdlib.h>")
    S("#include <mutex>")
    S("#define ME_STATIC_MAX_DEVICES 64")
    S("#define ME_SHARE_SLICE 524288L     // events per launch of the sharing kernel (%d KB of scratch per CTA in FP64)" % (NSCVEC * 8 * block * 8 // 1024))
    S("namespace me {")
    for gname, tmpl, rows in groups:
        nf = len(tmpl.params)
        # fully unrolled shapes: `static const`, so that every entry folds into an immediate; looped shapes: __constant__
        # (uniform-index reads through the constant cache instead of a global load in front of every shared-memory access)
        looped = UNROLL.get(gname, 1) < len(rows)
        S("%s int tab_%s_%s[%d][%d] = {" % ("__constant__" if looped else "static __device__ const", name, gname, len(rows), nf))
        for r in rows:
            S("  {%s}," % ", ".join(str(v) for v in r))
        S("};")
    S("// TM: slots >= %d (gluon-pair currents, row currents, jamps) live in tensor memory, %d columns per CTA: two CTAs per SM in FP64" % (lay.TM0, lay.tm_cols))
    S("// SH: current sharing across helicities (include/me.h ME_OPT_SHARE_CURRENTS): hels is in walk order (reflected Gray code, quark helicities")
    S("// fastest); a current whose own helicities did not change since the previous step is not re-evaluated (pairs, one-gluon quark currents:")
    S("// their slots still hold it; three-gluon sub-trees: reloaded from the L2-resident scratch `scratch`, %d vectors per thread)" % NSCVEC)
    S("template <typename R, typename RC, bool TM, bool SH, bool SEG = false>")
    S("__global__ void __launch_bounds__(%d) k_%s(const double* __restrict__ mom, long n, long npad, const unsigned char* __restrict__ hels, int nhel,"
      " double mt_d, double norm_hel, double inv_avg, double* __restrict__ me_out, double* __restrict__ me_hel, double* __restrict__ jamp_out,"
      " const int* __restrict__ helpe, void* __restrict__ scratch, double* __restrict__ part) {" % (block, name))
    S("  extern __shared__ __align__(16) unsigned char smem_raw[];")
    S("  R* sm = reinterpret_cast<R*>(smem_raw) + 2 * threadIdx.x;")
    S("  const long e0 = (long)blockIdx.x * blockDim.x + threadIdx.x;")
    S("  if (!TM && e0 >= npad) return;")
    S("  const long e = e0 < npad ? e0 : npad - 1;      // TMEM kernel: whole CTA stays (tcgen05 alloc / dealloc are CTA-wide); tail lanes repeat the last event")
    S("  uint32_t tm = 0, tm_base = 0;")
    S("  if constexpr (TM) {")
    S("    static_assert(sizeof(R) == 8 && ME_SM_STRIDE == 128, \"TMEM scratchpad: FP64, 128 threads per CTA\");")
    S("    __shared__ uint32_t tm_slot;")
    S("    tm_base = tm_alloc(&tm_slot, %d);" % lay.tm_cols)
    S("    tm = tm_base + ((uint32_t)(threadIdx.x & 96) << 16);      // this warp's quarter of the 128 lanes")
    S("  }")
    S("  const R mt = (R)mt_d;")
    S("  SpinorBasis<R> sbt, sbtb;")
    S("  {")
    S("    const double* pm = mom + (e >> 5) * (%d * 4 * 32) + (e & 31);" % NPAR)
    for k in range(NPAR):
        S("    const P4<double> pd%d = {pm[%d], pm[%d], pm[%d], pm[%d]};" % (k, (4 * k) * 32, (4 * k + 1) * 32, (4 * k + 2) * 32, (4 * k + 3) * 32))
    fixed = 0
    lines, fl = dd_invariant_lines(range(N), range(N), sgn, part)      # exact invariants (hel_amp.cuh "Propagator denominators")
    for l in lines:
        S("    " + l)
    fixed += fl
    for l in range(N):
        S("    stp<R>(sm, %d, pcast<R>(%s));" % (lay.MOM + 4 * l, "pd%d" % part(l) if sgn(l) > 0 else "pneg(pd%d)" % part(l)))
    S("    stp<R>(sm, %d, pcast<R>(pd2));" % lay.PT)
    for m, slot in lay.IK2.items():
        e, fl = dd_k2([i for i in range(N) if m >> i & 1], sgn)
        S("    sm[ME_EO(%d)] = (R)(1.0 / dd_value(%s));" % (slot, e)); fixed += fl + 2
    for m, slot in lay.IQ.items():
        e, fl = dd_q2([i for i in range(N) if m >> i & 1], sgn)
        S("    sm[ME_EO(%d)] = (R)(1.0 / dd_value(%s));" % (slot, e)); fixed += fl + 2
    for l in range(N):
        S("    { GluonBasis<R> gb = gluon_basis(pcast<R>(pd%d)); gb.bx *= (R)%d; gb.by *= (R)%d; stgb<R>(sm, %d, gb); }" % (part(l), -sgn(l), -sgn(l), lay.GBS[l]))
        fixed += 22
    S("    sbt = spinor_basis(pcast<R>(pd2), mt);")
    S("    sbtb = spinor_basis(pcast<R>(pd3), mt);")
    fixed += 40
    if PARK_SB:
        S("    // tensor-memory kernels: the two spinor bases are parked in the shared memory behind the %d slots (slots >= %d are tensor memory" % (lay.TM0, lay.TM0))
        S("    // there) and reloaded at the top of every step instead of holding 20 registers across the helicity walk")
        S("    if constexpr (TM) { stsb<R>(sm + ME_EO(%d), sbt); stsb<R>(sm + ME_EO(%d), sbtb); }" % (lay.TM0, lay.TM0 + 6))
    S("  }")
    S("  R* sc = nullptr;")
    S("  if constexpr (SH) sc = reinterpret_cast<R*>(scratch) + ((size_t)((SEG ? blockIdx.y * gridDim.x : 0u) + blockIdx.x) * (%d * 8 * ME_SM_STRIDE) + 2 * threadIdx.x);" % NSCVEC)
    S("  double acc = 0;")
    S("  int hprev = -1;")
    S("  // small batches: gridDim.y CTAs share the helicity list of an event block, each its own contiguous segment (the walk restarts with a")
    S("  // full evaluation); the |M|^2 of every step goes to part[step][event] and k_sum_steps adds them in list order: the same sequence of")
    S("  // additions as the loop below makes for gridDim.y = 1, so the result does not depend on the split, bit for bit")
    S("  // (SEG = false: the kernel of the large batches, one segment, no per-step buffer: nothing of this costs it a register)")
    S("  int ih_begin = 0, ih_end = nhel;")
    S("  if constexpr (SEG) {")
    S("    const int seg_len = (nhel + (int)gridDim.y - 1) / (int)gridDim.y;")
    S("    ih_begin = (int)blockIdx.y * seg_len; ih_end = ih_begin + seg_len < nhel ? ih_begin + seg_len : nhel;")
    S("  }")
    S("  for (int ih = ih_begin; ih < ih_end; ++ih) {")
    S("    const int h = helpe != nullptr ? helpe[e < n ? e : n - 1] : hels[ih];")
    S("    const int chg = (SH && hprev >= 0) ? (h ^ hprev) : %d;      // helicities that changed since the previous step" % ((1 << NPAR) - 1))
    S("    hprev = h;")
    if PARK_SB:
        S("    const W4<R> ub = spinor_ubar(TM ? ldsb<R>(sm + ME_EO(%d)) : sbt, lam_of<R>(h, %d));" % (lay.TM0, NPAR - 1 - 2))
        S("    const W4<R> vv = spinor_v(TM ? ldsb<R>(sm + ME_EO(%d)) : sbtb, lam_of<R>(h, %d));" % (lay.TM0 + 6, NPAR - 1 - 3))
    else:
        S("    const W4<R> ub = spinor_ubar(sbt, lam_of<R>(h, %d));" % (NPAR - 1 - 2))
        S("    const W4<R> vv = spinor_v(sbtb, lam_of<R>(h, %d));" % (NPAR - 1 - 3))
    S("    const W4<R> jtt = bilinear(ub, vv);")
    S("    if constexpr (TM) {")
    S("      const uint32_t zz[16] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};")
    S("#pragma unroll")
    S("      for (int s = 0; s < %d; ++s) tm_st16(tm + ME_TM_COL(R, ME_EO(%d)) + 16 * s, zz);" % (ncol // 4, lay.J))
    S("    } else {")
    S("#pragma unroll")
    S("      for (int s = 0; s < %d; ++s) cset<R>(sm + ME_EO(%d + 2 * s), (R)0, (R)0);" % (ncol, lay.J))
    S("    }")
    for gname, tmpl, rows in groups:
        S("    // ---- %s: %d instances" % (gname, len(rows)))
        if tmpl.mode != "both":
            S("    if constexpr (%sSH) {" % ("" if tmpl.mode == "sh" else "!"))
        if gname in UNROLL_SH:      # executed on few steps of the walk in the sharing kernel: a compact loop costs nothing there and keeps the body small
            S("#pragma unroll(sizeof(R) == 8 ? (SH ? %d : %d) : %d)" % (UNROLL_SH[gname], UNROLL.get(gname, 1), UNROLL32.get(gname, 1)))
        else:
            S("#pragma unroll(sizeof(R) == 8 ? %d : %d)" % (UNROLL.get(gname, 1), UNROLL32.get(gname, 1)))
        S("    for (int it = 0; it < %d; ++it) {" % len(rows))
        S("      const int* tb = tab_%s_%s[it];" % (name, gname))
        for l in tmpl.lines:
            S("      " + l)
        S("    }")
        if tmpl.mode != "both":
            S("    }")
    S("    RC cr[%d], ci[%d];" % (ncol, ncol))
    S("    if constexpr (TM) {")
    S("      XW<R, TM> jx[%d];" % (ncol // 4))
    S("      xwait_st<TM>();")
    S("#pragma unroll")
    S("      for (int s = 0; s < %d; ++s) xldw_issue<R, TM>(jx[s], sm, tm, ME_EO(%d + 8 * s));" % (ncol // 4, lay.J))
    S("#pragma unroll")
    S("      for (int s = 0; s < %d; ++s) {" % (ncol // 4))
    S("        const W4<R> w = xldw_get<R, TM>(jx[s]);")
    S("        if (jamp_out != nullptr && e0 < n) {")
    S("          const R v[8] = {w.r0, w.i0, w.r1, w.i1, w.r2, w.i2, w.r3, w.i3};")
    S("#pragma unroll")
    S("          for (int k = 0; k < 8; ++k) jamp_out[(long)(8 * s + k) * n + e0] = (double)v[k];")
    S("        }")
    S("        cr[4 * s] = (RC)w.r0; ci[4 * s] = (RC)w.i0; cr[4 * s + 1] = (RC)w.r1; ci[4 * s + 1] = (RC)w.i1;")
    S("        cr[4 * s + 2] = (RC)w.r2; ci[4 * s + 2] = (RC)w.i2; cr[4 * s + 3] = (RC)w.r3; ci[4 * s + 3] = (RC)w.i3;")
    S("      }")
    S("    } else {")
    S("      if (jamp_out != nullptr && e0 < n) {")
    S("#pragma unroll")
    S("        for (int s = 0; s < %d; ++s) jamp_out[(long)s * n + e0] = (double)sm[ME_EO(%d + s)];" % (2 * ncol, lay.J))
    S("      }")
    S("#pragma unroll")
    S("      for (int s = 0; s < %d; ++s) { R jr, ji; cget<R>(sm + ME_EO(%d + 2 * s), jr, ji); cr[s] = (RC)jr; ci[s] = (RC)ji; }" % (ncol, lay.J))
    S("    }")
    for l in cs_lines:
        S("    " + l)
    S("    const double meh = (double)cs;")
    S("    if (me_hel != nullptr && e0 < n) me_hel[(long)h * n + e0] = meh * norm_hel;")
    S("    if constexpr (SEG) { if (e0 < n) part[(long)ih * n + e0] = meh; }")
    S("    else acc += meh;")
    S("  }")
    S("  if constexpr (!SEG) { if (me_out != nullptr && e0 < n) me_out[e0] = acc * norm_hel * inv_avg; }")
    S("  if constexpr (TM) tm_free(tm_base, %d);" % lay.tm_cols)
    S("}")
    S("// sum over the steps of the helicity list in list order (see the kernel above)")
    S("static __global__ void k_sum_steps_%s(const double* __restrict__ part, int nhel, long n, double norm_hel, double inv_avg, double* __restrict__ me_out) {" % name)
    S("  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;")
    S("  if (e >= n) return;")
    S("  double acc = 0;")
    S("  for (int ih = 0; ih < nhel; ++ih) acc += part[(long)ih * n + e];")
    S("  me_out[e] = acc * norm_hel * inv_avg;")
    S("}")
    S("// segments of the helicity list per event block: as many as fill the CTA slots of the device (two per SM), at least %d steps each" % MIN_SEG_STEPS)
    S("static int segments_%s(long npad, int nhel, int nsm) {" % name)
    S("  const long ctas = (npad + %d - 1) / %d;" % (block, block))
    S("  long s = (2L * nsm) / ctas;")
    S("  if (s > nhel / %d) s = nhel / %d;" % (MIN_SEG_STEPS, MIN_SEG_STEPS))
    S("  return s < 1 ? 1 : (int)s;")
    S("}")
    S("// bytes of the current cache: one region per CTA, nseg segments per event block (0: kernel without sharing, no cache)")
    S("static size_t cache_bytes_%s(int precision, long npad, int nseg) {" % name)
    S("  const long np = npad < ME_SHARE_SLICE ? npad : ME_SHARE_SLICE;")
    S("  return (size_t)((np + %d - 1) / %d) * nseg * %d * 8 * %d * (precision == 2 ? sizeof(float) : sizeof(double));" % (block, block, NSCVEC, block))
    S("}")
    S("static cudaError_t launch_%s(int precision, const LaunchArgs& a) {" % name)
    S("  const unsigned grid = (unsigned)((a.npad + %d - 1) / %d);" % (block, block))
    S("  const size_t smd = sizeof(double) * %d * %d, smf = sizeof(float) * %d * %d, smt = sizeof(double) * %d * %d;" % (lay.nslots, block, lay.nslots, block, lay.TM0 + (12 if PARK_SB else 0), block))
    S("  // FP64 amplitudes (double and mixed): tensor-memory kernel, two CTAs per SM; ME_NO_TMEM=1 selects the shared-memory-only kernel (A/B timing)")
    S("  static const bool no_tmem = getenv(\"ME_NO_TMEM\") != nullptr && getenv(\"ME_NO_TMEM\")[0] == '1';")
    S("  const bool sh = a.share != 0 && a.hel_per_event == nullptr && a.scratch != nullptr && !no_tmem && a.me_hel == nullptr && a.jamp_out == nullptr && a.me_out != nullptr;")
    S("  // small batch, only me_out wanted: split the helicity list over gridDim.y (the per-step buffer sits behind the current cache in a.scratch)")
    S("  const bool only_me = a.hel_per_event == nullptr && a.me_hel == nullptr && a.jamp_out == nullptr && a.me_out != nullptr;")
    S("  const int nseg = (only_me && sh) ? segments_%s(a.npad, a.nhel, a.nsm) : 1;" % name)
    S("  double* part = nullptr;")
    S("  if (nseg > 1) {")
    S("    const size_t off = (cache_bytes_%s(precision, a.npad, nseg) + 255) / 256 * 256;" % name)
    S("    if (a.scratch_bytes < off + sizeof(double) * (size_t)a.nhel * a.n) return cudaErrorInvalidValue;")
    S("    part = reinterpret_cast<double*>((char*)a.scratch + off);")
    S("  }")
    S("  const dim3 grid2(grid, (unsigned)nseg);")
    S("#define ME_ARGS a.mom, a.n, a.npad, a.hels, a.nhel, a.mt, a.norm_hel, a.inv_avg, a.me_out, a.me_hel, a.jamp_out, a.hel_per_event, a.scratch, part")
    S("#define ME_LAUNCH(K, SMEM) do { cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM)); \\")
    S("    cudaFuncSetAttribute(K, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared); \\")
    S("    K<<<grid2, %d, SMEM, a.stream>>>(ME_ARGS); } while (0)" % block)
    S("  if (sh) {       // slices of at most ME_SHARE_SLICE events, one after the other on the stream: the scratch (one region per CTA) stays bounded")
    S("    for (long start = 0; start < a.npad; start += ME_SHARE_SLICE) {")
    S("      const long np = a.npad - start < ME_SHARE_SLICE ? a.npad - start : ME_SHARE_SLICE, nn = a.n - start < np ? a.n - start : np;")
    S("      const dim3 sgrid((unsigned)((np + %d - 1) / %d), (unsigned)nseg);      // (nseg > 1 only for batches far below one slice)" % (block, block))
    S("#define ME_SARGS a.mom + (start / ME_PAGE) * (%d * 4 * ME_PAGE), nn, np, a.hels, a.nhel, a.mt, a.norm_hel, a.inv_avg, a.me_out + start, nullptr, nullptr, nullptr, a.scratch, part" % NPAR)
    S("#define ME_SLAUNCH(K, SMEM) do { cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM)); \\")
    S("    cudaFuncSetAttribute(K, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared); \\")
    S("    K<<<sgrid, %d, SMEM, a.stream>>>(ME_SARGS); } while (0)" % block)
    S("      if (nseg > 1) {")
    S("        if (precision == 0) ME_SLAUNCH((k_%s<double, double, true, true, true>), smt);" % name)
    S("        else if (precision == 1) ME_SLAUNCH((k_%s<double, float, true, true, true>), smt);" % name)
    S("        else ME_SLAUNCH((k_%s<float, float, false, true, true>), smf);" % name)
    S("      } else if (precision == 0) ME_SLAUNCH((k_%s<double, double, true, true>), smt);" % name)
    S("      else if (precision == 1) ME_SLAUNCH((k_%s<double, float, true, true>), smt);" % name)
    S("      else ME_SLAUNCH((k_%s<float, float, false, true>), smf);" % name)
    S("#undef ME_SLAUNCH")
    S("#undef ME_SARGS")
    S("    }")
    S("  } else if (precision == 0) {")
    S("    if (no_tmem) ME_LAUNCH((k_%s<double, double, false, false>), smd); else ME_LAUNCH((k_%s<double, double, true, false>), smt);" % (name, name))
    S("  } else if (precision == 1) {")
    S("    if (no_tmem) ME_LAUNCH((k_%s<double, float, false, false>), smd); else ME_LAUNCH((k_%s<double, float, true, false>), smt);" % (name, name))
    S("  } else {")
    S("    ME_LAUNCH((k_%s<float, float, false, false>), smf);" % name)
    S("  }")
    S("#undef ME_LAUNCH")
    S("#undef ME_ARGS")
    S("  if (nseg > 1) k_sum_steps_%s<<<(unsigned)((a.n + 255) / 256), 256, 0, a.stream>>>(part, a.nhel, a.n, a.norm_hel, a.inv_avg, a.me_out);" % name)
    S("  return cudaGetLastError();")
    S("}")
    # ---- the sharing kernel on a scratch that nobody allocates (include/me.h me_compute_static): a file-scope device array of a fixed size
    static_ctas = STATIC_MAX_EVENTS // block
    S("// Sharing kernel without any allocation: its current cache is this file-scope array (%d CTAs x %d vectors x 8 x %d threads of double:" % (static_ctas, NSCVEC, block))
    S("// %.1f MiB that every GPU which loads the library holds until exit).  In host code the NAME of the array is a host-side stand-in, not" % (static_ctas * NSCVEC * 8 * block * 8 / 2.0 ** 20))
    S("// a device address: the launcher below asks the runtime for the address once per device, with that device current.")
    S("static __device__ __align__(256) unsigned char static_scratch_%s[%dUL * %d * 8 * %d * sizeof(double)];" % (name, static_ctas, NSCVEC, block))
    S("extern const long static_max_events_%s = %dL;" % (name, STATIC_MAX_EVENTS))
    S("cudaError_t launch_%s_static(int precision, const LaunchArgs& a) {" % name)
    S("  if (a.npad > %dL || a.me_out == nullptr || a.hel_per_event != nullptr) return cudaErrorInvalidValue;" % STATIC_MAX_EVENTS)
    S("  static void* addr[ME_STATIC_MAX_DEVICES];         // device address of the array on every device seen so far")
    S("  static std::mutex mtx;")
    S("  int dev = -1;")
    S("  cudaError_t e = cudaGetDevice(&dev);")
    S("  if (e != cudaSuccess) return e;")
    S("  if (dev < 0 || dev >= ME_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;")
    S("  void* ptr = nullptr;")
    S("  {")
    S("    std::lock_guard<std::mutex> lock(mtx);")
    S("    if (addr[dev] == nullptr) {                      // set-up, once per device")
    S("      e = cudaGetSymbolAddress((void**)&addr[dev], static_scratch_%s);" % name)
    S("      if (e != cudaSuccess) { addr[dev] = nullptr; return e; }")
    S("    }")
    S("    ptr = addr[dev];")
    S("  }")
    S("  // nothing in the array has to start at zero: the first step of the helicity walk writes every vector before any step reads it")
    S("  const unsigned grid = (unsigned)((a.npad + %d - 1) / %d);" % (block, block))
    S("  const size_t smf = sizeof(float) * %d * %d, smt = sizeof(double) * %d * %d;" % (lay.nslots, block, lay.TM0 + (12 if PARK_SB else 0), block))
    S("#define ME_TARGS a.mom, a.n, a.npad, a.hels, a.nhel, a.mt, a.norm_hel, a.inv_avg, a.me_out, nullptr, nullptr, nullptr, ptr, nullptr")
    S("#define ME_TLAUNCH(K, SMEM) do { cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM)); \\")
    S("    cudaFuncSetAttribute(K, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared); \\")
    S("    K<<<grid, %d, SMEM, a.stream>>>(ME_TARGS); } while (0)" % block)
    S("  if (precision == 0) ME_TLAUNCH((k_%s<double, double, true, true>), smt);" % name)
    S("  else if (precision == 1) ME_TLAUNCH((k_%s<double, float, true, true>), smt);" % name)
    S("  else if (precision == 2) ME_TLAUNCH((k_%s<float, float, false, true>), smf);" % name)
    S("  else return cudaErrorInvalidValue;")
    S("#undef ME_TLAUNCH")
    S("#undef ME_TARGS")
    S("  return cudaGetLastError();")
    S("}")
    S("static const double color_num_%s[%d] = {%s};" % (name, ncol * ncol, ", ".join(str(float(x)) for row in color_num for x in row)))
    # current sharing: scratch of one CTA = NSCVEC vectors x 8 reals x threads; rank of every helicity in the walk; algorithmic flops per event
    walk = gray_walk()
    rank = [walk.index(h) for h in range(1 << NPAR)]
    S("static const unsigned char gray_rank_%s[%d] = {%s};" % (name, 1 << NPAR, ", ".join(str(r) for r in rank)))
    S("// current cache (sharing on) + for small batches the per-step buffer of the helicity-segment split, sized for the full helicity list")
    S("static size_t scratch_%s(int precision, long npad, int share, int nsm) {" % name)
    S("  if (!share) return 0;")
    S("  const int nseg = segments_%s(npad, %d, nsm);" % (name, 1 << NPAR))
    S("  const size_t cache = cache_bytes_%s(precision, npad, nseg);" % name)
    S("  return nseg > 1 ? (cache + 255) / 256 * 256 + sizeof(double) * %d * (size_t)npad : cache;" % (1 << NPAR))
    S("}")
    nh = 1 << NPAR
    shared = 0
    for _, t, rows in groups:
        if t.mode == "plain":
            continue
        for conds in t.cond_all:
            always = t.flops - sum(f for _, f in conds)
            shared += always * nh + sum(f * walk_count(m, walk) for m, f in conds)
    shared_event = shared + nh * (cs_flops + 2 * FL["spinor"] + FL["bilinear"]) + fixed
    S("extern const ProcTable tab_%s = {%d, %d, %d, %d, %d, 1, {%r, %r, %r}, {%r, %r, %r}, %r, color_num_%s, launch_%s, scratch_%s, false, gray_rank_%s, %r, 0, 0.0};"
      % (name, N, 123, namp, ncol, color_denom, float(per_hel), float(per_hel), float(per_hel),
         float(per_hel), float(per_hel), float(per_hel), float(fixed), name, name, name, name, float(shared_event)))
    S("}  // namespace me")
    info = dict(n=N, ndiagrams=123, namp=namp, ncol=ncol, color_denom=color_denom, flops_per_helicity=per_hel,
                flops_executed_per_helicity=per_hel, fixed_flops=fixed, flops_shared_event=shared_event, gray_walk=walk, colour_flops=cs_flops, smem_slots=lay.nslots, tm_slot0=lay.TM0, tm_cols=lay.tm_cols, block=block,
                shapes={g: len(r) for g, t, r in groups if t.mode != "sh"}, color_num=color_num)
    return "\n".join(src) + "\n", info
