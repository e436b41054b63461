"""Colour-ordered (Berends-Giele) recursion for the partial amplitudes of g g -> t t~ + (n-2) g: a third, independent route to the
colour-flow amplitudes ("jamps"; the check suggested at SURVEY.md line 408).

    M_{i k}(colours) = sum over the n! orderings s of  (T^{s(1)} ... T^{s(n)})_{i k}  A(s)

Test infrastructure: numpy only, explicit 4x4 gamma matrices, external states from their defining equations (tests/brute_force.py).
No diagram list and no colour algebra at run time: the ordered vertices below are the Feynman rules of SURVEY.md section 8(c) C1-C3
with f^{abc} T^c = -i [T^a, T^b] substituted once, by hand:

  * three-gluon vertex  g f^{abc} V3(1,2)  ->  ordered pair (L, R):  -i g V3(J_L, J_R)   (V3 is antisymmetric in its two legs, so
    the term with the commutator's other order is the same expression for the split (R, L));
  * four-gluon vertex  -i g^2 [f^{abe}f^{cde}(..) + f^{ace}f^{bde}(..) + f^{ade}f^{bce}(..)] with f f T = -[[.,.],.]  ->  ordered
    triple (L, M, R):  -i g^2 [ (J_L.J_M) J_R + (J_M.J_R) J_L - 2 (J_L.J_R) J_M ];
  * quark line from the outgoing t: the gluon blocks of an ordering are attached in order, vertex i g gamma^mu, propagator
    i (qslash + m) / (q^2 - m^2), and the colour string is the product of the T's in the order of attachment.

The amplitudes carry every factor of the full rules (g_s^n and all i's); the library strips g_s^n and a global phase from its jamps
(DESIGN.md "Normalisation"), so the tests compare up to ONE complex constant per process, the same for all orderings, helicities and
events, whose modulus must be g_s^n.
"""
import itertools

import numpy as np

from brute_force import GAM, GS, I4, METRIC, PRM, def_eps, def_u, def_v, gell_mann, slash


def mdot(a, b):
    return a @ METRIC @ b


def ordered_amplitudes(n, p, hel):
    """{ordering (tuple of gluon labels 0..n-1, first = attached next to the t): A(ordering)} for one event p[npar][4] and
    helicities hel[npar] (+-1).  Gluon labels: 0, 1 = the incoming beams, 2.. = the final-state gluons."""
    mt = PRM["mt"]
    part = lambda g: g if g < 2 else g + 2
    sgn = lambda g: 1 if g < 2 else -1
    eps = {}
    for g in range(n):
        e = def_eps(p[part(g)], hel[part(g)])
        eps[g] = e if g < 2 else e.conj()
    K = lambda blk: sum((sgn(g) * p[part(g)] for g in blk), np.zeros(4))

    def v3(J1, k1, J2, k2):
        """kinematic bracket of the three-gluon vertex, legs 1, 2 incoming with momenta k1, k2, open index up"""
        k3 = -(k1 + k2)
        return mdot(J1, J2) * (k1 - k2) + mdot(k2 - k3, J1) * J2 + mdot(k3 - k1, J2) * J1

    cur = {}

    def J(blk):                                   # ordered off-shell gluon current of the block, propagator included
        if blk in cur:
            return cur[blk]
        if len(blk) == 1:
            cur[blk] = eps[blk[0]]
            return cur[blk]
        acc = np.zeros(4, complex)
        for i in range(1, len(blk)):
            L, R = blk[:i], blk[i:]
            acc = acc + (-1j * GS) * v3(J(L), K(L), J(R), K(R))
        for i in range(1, len(blk) - 1):
            for j in range(i + 1, len(blk)):
                JL, JM, JR = J(blk[:i]), J(blk[i:j]), J(blk[j:])
                acc = acc + (-1j * GS ** 2) * (mdot(JL, JM) * JR + mdot(JM, JR) * JL - 2 * mdot(JL, JR) * JM)
        k = K(blk)
        cur[blk] = (-1j / mdot(k, k)) * acc
        return cur[blk]

    pt, ptb = p[2], p[3]
    ub = def_u(pt, mt, hel[2]).conj() @ GAM[0]
    v = def_v(ptb, mt, hel[3])
    line = {(): ub}

    def psi(lst):                                 # row spinor: ubar with the gluons of lst attached in order, propagator included
        if lst in line:
            return line[lst]
        q = pt - K(lst)
        prop = 1j * (slash(q) + mt * I4) / (mdot(q, q) - mt ** 2)
        acc = np.zeros(4, complex)
        for i in range(len(lst)):
            acc = acc + (1j * GS) * (psi(lst[:i]) @ slash(J(lst[i:]))) @ prop
        line[lst] = acc
        return acc

    out = {}
    for s in itertools.permutations(range(n)):
        a = 0
        for i in range(n):
            a = a + (1j * GS) * (psi(s[:i]) @ slash(J(s[i:]))) @ v
        out[s] = a
    return out


def colour_matrix(n):
    """C[s][t] = sum over quark colours of (T^{s(1)}..T^{s(n)})_{ik} conj((T^{t(1)}..T^{t(n)})_{ik}), summed over the gluon colours: the
    numeric colour matrix in the basis of ordered_amplitudes, from explicit Gell-Mann matrices (for n <= 4: 8^n terms)"""
    T = gell_mann()
    perms = list(itertools.permutations(range(n)))
    strings = []
    for s in perms:
        # tensor [colour of gluon 0, .., colour of gluon n-1, i, k]
        letters = "abcdefgh"[:n]
        ops = [T] * n
        idx = "ij"
        expr = []
        prev = "i"
        for pos, g in enumerate(s):
            nxt = "k" if pos == n - 1 else "xyzwv"[pos]
            expr.append(letters[g] + prev + nxt)
            prev = nxt
        strings.append(np.einsum(",".join(expr) + "->" + letters + "ik", *ops))
    C = np.zeros((len(perms), len(perms)), complex)
    for a, A in enumerate(strings):
        for b, B in enumerate(strings):
            C[a, b] = np.vdot(B, A)
    return perms, C
