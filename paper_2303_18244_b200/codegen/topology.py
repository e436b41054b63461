"""Build-time diagram enumeration and colour algebra for g g -> t t~ + (n-2) g.

Product code (the CUDA generator's front end) — independent of oracle/: exact integer /
Fraction arithmetic, colour matrix from the Fierz identity (no numeric Gell-Mann matrices).

Feynman rules restated in DESIGN.md (PAPER.md has no formulas).
Every gluon sub-tree ("G term") and partial quark line ("Q term") is an off-shell current with
the factors of i and g_s *stripped*; the phase i^k is folded into the colour polynomial of the
term, so the jamp coefficients c_{d,sigma} come out as Gaussian integers in {0,+-1,+-i}.

Gluon labels 0..n-1: 0,1 = incoming (particles 0,1), 2.. = outgoing (particles 4,5,..).
Colour basis: strings T^{a_s(0)}...T^{a_s(n-1)} (t colour index left, t~ right), s running over
the permutations of the labels in lexicographic order -> ncol = n!.
"""
from fractions import Fraction
from itertools import permutations

I = 1j


def _pmul(a, b):
    r = {}
    for sa, ca in a.items():
        for sb, cb in b.items():
            s = sa + sb
            r[s] = r.get(s, 0) + ca * cb
    return r


def _padd(a, b, cb=1):
    r = dict(a)
    for s, c in b.items():
        r[s] = r.get(s, 0) + cb * c
    return {s: c for s, c in r.items() if c != 0}


def _pscale(a, c):
    return {s: c * v for s, v in a.items()}


def _pcomm(a, b):
    return _padd(_pmul(a, b), _pmul(b, a), -1)


class GTerm:
    """One gluon sub-tree with one colour structure.  kind: 'leaf' | 'v3' | 'v4_0' | 'v4_1' | 'v4_2'."""
    __slots__ = ("id", "mask", "kind", "ch", "col", "canon", "size")

    def __init__(self, id, mask, kind, ch, col, canon):
        self.id, self.mask, self.kind, self.ch, self.col, self.canon = id, mask, kind, ch, col, canon
        self.size = bin(mask).count("1")


class QTerm:
    """Partial quark line grown from the outgoing t: prev (QTerm id or -1 for the bare ubar) + attached GTerm."""
    __slots__ = ("id", "mask", "prev", "g", "col", "canon", "size")

    def __init__(self, id, mask, prev, g, col, canon):
        self.id, self.mask, self.prev, self.g, self.col, self.canon = id, mask, prev, g, col, canon
        self.size = bin(mask).count("1")


class Closure:
    """Amplitude  qbar(q) . Vslash(g) . v(t~);  jamp = [(colour index, Gaussian-integer coefficient)]."""
    __slots__ = ("id", "q", "g", "jamp", "canon")

    def __init__(self, id, q, g, jamp, canon):
        self.id, self.q, self.g, self.jamp, self.canon = id, q, g, jamp, canon


def _submasks_with_low(m):
    """proper non-empty submasks of m that contain m's lowest set bit"""
    low = m & -m
    a = (m - 1) & m
    while a:
        if a & low:
            yield a
        a = (a - 1) & m


class Topology:
    def __init__(self, n):
        self.n = n
        full = (1 << n) - 1
        self.full = full
        G, Gby = [], {m: [] for m in range(1, full + 1)}
        masks = sorted(range(1, full + 1), key=lambda m: (bin(m).count("1"), m))
        for m in masks:
            if m & (m - 1) == 0:
                lab = m.bit_length() - 1
                t = GTerm(len(G), m, "leaf", (), {(lab,): 1}, True)
                G.append(t); Gby[m].append(t.id)
                continue
            # three-gluon vertex, unordered split {A,B}, A holds the lowest label.
            # stripped current: kin3/K^2 ; phase (-i)_prop * colour f -> -i[X1,X2]  => col = -[X1,X2]
            for A in _submasks_with_low(m):
                B = m ^ A
                for a in Gby[A]:
                    for b in Gby[B]:
                        col = _pscale(_pcomm(G[a].col, G[b].col), -1)
                        t = GTerm(len(G), m, "v3", (a, b), col, G[a].canon and G[b].canon)
                        G.append(t); Gby[m].append(t.id)
            # four-gluon vertex, unordered split {A,B,C}: A holds the lowest label, B the lowest of the rest.
            # vertex -i g^2 [ f^{abe}f^{cde}(..) + f^{ace}f^{bde}(..) + f^{ade}f^{bce}(..) ], prop -i:
            # phase (-i)(-i) = -1 times colour  -[[X1,X2],X3], -[[X1,X3],X2], +[X1,[X2,X3]]
            for A in _submasks_with_low(m):
                rest = m ^ A
                for B in _submasks_with_low(rest):
                    C = rest ^ B
                    for a in list(Gby[A]):
                        for b in list(Gby[B]):
                            for c in list(Gby[C]):
                                X1, X2, X3 = G[a].col, G[b].col, G[c].col
                                cols = (_pcomm(_pcomm(X1, X2), X3), _pcomm(_pcomm(X1, X3), X2),
                                        _pscale(_pcomm(X1, _pcomm(X2, X3)), -1))
                                can = G[a].canon and G[b].canon and G[c].canon
                                for k in range(3):
                                    t = GTerm(len(G), m, "v4_%d" % k, (a, b, c), cols[k], can and k == 0)
                                    G.append(t); Gby[m].append(t.id)
        self.G, self.Gby = G, Gby
        # quark line: psibar' = psibar (i g Vslash) i(qslash+m)/(q^2-m^2) -> phase i*i = -1
        Q, Qby = [], {m: [] for m in range(0, full + 1)}
        for m in masks:
            if m == full:
                continue
            a = m
            while a:
                s = m ^ a
                prevs = Qby[s] if s else [-1]
                for q in prevs:
                    for g in Gby[a]:
                        qcol = Q[q].col if q >= 0 else {(): 1}
                        col = _pscale(_pmul(qcol, G[g].col), -1)
                        can = (Q[q].canon if q >= 0 else True) and G[g].canon
                        t = QTerm(len(Q), m, q, g, col, can)
                        Q.append(t); Qby[m].append(t.id)
                a = (a - 1) & m
        self.Q, self.Qby = Q, Qby
        # colour basis and closures: amplitude  psibar (i g Vslash) v  -> phase i
        self.perms = list(permutations(range(n)))
        self.perm_index = {p: i for i, p in enumerate(self.perms)}
        self.ncol = len(self.perms)
        Cl = []
        for s in range(0, full):
            a = full ^ s
            prevs = Qby[s] if s else [-1]
            for q in prevs:
                for g in Gby[a]:
                    qcol = Q[q].col if q >= 0 else {(): 1}
                    col = _pscale(_pmul(qcol, G[g].col), I)
                    jamp = []
                    for st, c in sorted(col.items()):
                        if c == 0:
                            continue
                        assert c in (1, -1, 1j, -1j), c
                        jamp.append((self.perm_index[st], complex(c)))
                    can = (Q[q].canon if q >= 0 else True) and G[g].canon
                    Cl.append(Closure(len(Cl), q, g, jamp, can))
        self.Cl = Cl
        self.ndiagrams = sum(1 for c in Cl if c.canon)
        self.color_num, self.color_denom = color_matrix(self.perms)


# ------------------------------------------------------------------------------------------
# Colour matrix  C_{s t} = sum_{a_1..a_n} Tr( T^{s} (T^{t})^dagger ),  exactly, by the Fierz identity
#   T^a_{ij} T^a_{kl} = 1/2 ( d_il d_jk - 1/N d_ij d_kl )      (Tr T^a T^b = d^{ab}/2, N = 3)
# ------------------------------------------------------------------------------------------
NC = 3


def _trace_product(words):
    """sum over all colour indices of prod_w Tr(T^{w[0]} T^{w[1]} ...); every label occurs exactly twice overall."""
    words = [tuple(w) for w in words]
    for wi, w in enumerate(words):
        if not w:
            continue
        a = w[0]
        rest = list(words[:wi] + words[wi + 1:])
        if a in w[1:]:
            j = w.index(a, 1)
            Y, Z = w[1:j], w[j + 1:]
            # Tr(T^a Y T^a Z) = 1/2 [ Tr(Y) Tr(Z) - 1/N Tr(Y Z) ]
            return Fraction(1, 2) * (_trace_product(rest + [Y, Z]) - Fraction(1, NC) * _trace_product(rest + [Y + Z]))
        for wj, w2 in enumerate(rest):
            if a in w2:
                j = w2.index(a)
                Y = w[1:]
                Z = w2[j + 1:] + w2[:j]
                others = rest[:wj] + rest[wj + 1:]
                # Tr(T^a Y) Tr(T^a Z) = 1/2 [ Tr(Y Z) - 1/N Tr(Y) Tr(Z) ]
                return Fraction(1, 2) * (_trace_product(others + [Y + Z]) - Fraction(1, NC) * _trace_product(others + [Y, Z]))
        raise AssertionError("unpaired colour label")
    r = Fraction(1)
    for _ in words:
        r *= NC          # Tr(1) = N for every emptied trace
    return r


def color_matrix(perms):
    """Returns (integer numerators [ncol][ncol], common denominator)."""
    n = len(perms[0])
    ident = tuple(range(n))
    index = {p: i for i, p in enumerate(perms)}
    row = [_trace_product([ident + tuple(reversed(p))]) for p in perms]
    denom = 1
    for f in row:
        denom = denom * f.denominator // _gcd(denom, f.denominator)
    num_row = [int(f * denom) for f in row]
    ncol = len(perms)
    C = [[0] * ncol for _ in range(ncol)]
    for s, ps in enumerate(perms):
        inv = [0] * n
        for k, lab in enumerate(ps):
            inv[lab] = k
        for t, pt in enumerate(perms):
            rel = tuple(inv[lab] for lab in pt)
            C[s][t] = num_row[index[rel]]
    return C, denom


def _gcd(a, b):
    while b:
        a, b = b, a % b
    return a
