"""Brute-force definition of sum_colours |M(p, h, colours)|^2 for g g -> t t~ + (n-2) g, used as a pin that has NO diagram
list and NO colour-flow basis (tests/test_oracle_me.py pins the oracle with it; tests/test_gpu_parity.py compares the CUDA
path with it directly, so that the oracle's diagram enumerator is not on the chain between the GPU and an independent
definition).  Test infrastructure: numpy only, explicit 4x4 gamma matrices, explicit f^{abc} and T^a_{ij}; external states
from their defining eigenvalue equations.  Feynman rules: SURVEY.md section 8(c) C1-C3 (PAPER.md prints none: P:20)."""
import math

import numpy as np

PRM = dict(mz=91.188, wz=2.441404, aewm1=132.507, sw2=0.2222, mt=173.0, alpha_s=0.118)
GS = math.sqrt(4 * math.pi * PRM["alpha_s"])

# ---------------------------------------------------------------- explicit Dirac algebra (chiral basis)
S0 = np.eye(2, dtype=complex)
SIG = [np.array([[0, 1], [1, 0]], complex), np.array([[0, -1j], [1j, 0]], complex), np.array([[1, 0], [0, -1]], complex)]
Z2 = np.zeros((2, 2), complex)
GAM = np.array([np.block([[Z2, S0], [S0, Z2]])] + [np.block([[Z2, s], [-s, Z2]]) for s in SIG])   # gamma^mu
METRIC = np.diag([1.0, -1.0, -1.0, -1.0])
SIGMA3 = [np.block([[s, Z2], [Z2, s]]) for s in SIG]                                               # spin operator
I4 = np.eye(4, dtype=complex)


def slash(v):
    return sum(METRIC[m, m] * v[m] * GAM[m] for m in range(4))


def null_vector(M):
    _, s, vh = np.linalg.svd(M)
    assert s[-1] < 1e-9 * s[0]
    return vh[-1].conj()


def def_u(p, m, lam):
    """u(p,lam) from its defining equations: (pslash - m)u = 0, (Sigma.phat)u = lam u, u^dag u = 2E."""
    ph = p[1:] / np.linalg.norm(p[1:])
    hel = sum(ph[i] * SIGMA3[i] for i in range(3))
    u = null_vector(np.vstack([slash(p) - m * I4, (hel - lam * I4) * p[0]]))
    return u * math.sqrt(2 * p[0]) / np.linalg.norm(u)


def def_v(p, m, lam):
    """v(p,lam): (pslash + m)v = 0, (Sigma.phat)v = -lam v (lam = physical antiparticle helicity), v^dag v = 2E."""
    ph = p[1:] / np.linalg.norm(p[1:])
    hel = sum(ph[i] * SIGMA3[i] for i in range(3))
    v = null_vector(np.vstack([slash(p) + m * I4, (hel + lam * I4) * p[0]]))
    return v * math.sqrt(2 * p[0]) / np.linalg.norm(v)


def def_eps(p, lam):
    """eps(p,lam): eps^0 = 0, eps.p = 0, i phat x eps = lam eps, |eps| = 1."""
    ph = p[1:] / np.linalg.norm(p[1:])
    cross = np.array([[0, -ph[2], ph[1]], [ph[2], 0, -ph[0]], [-ph[1], ph[0], 0]], complex)
    e = null_vector(np.vstack([1j * cross - lam * np.eye(3), ph[None, :]]))
    return np.concatenate([[0], e / np.linalg.norm(e)])



def gell_mann():
    l = np.zeros((8, 3, 3), complex)
    l[0][0, 1] = l[0][1, 0] = 1
    l[1][0, 1], l[1][1, 0] = -1j, 1j
    l[2][0, 0], l[2][1, 1] = 1, -1
    l[3][0, 2] = l[3][2, 0] = 1
    l[4][0, 2], l[4][2, 0] = -1j, 1j
    l[5][1, 2] = l[5][2, 1] = 1
    l[6][1, 2], l[6][2, 1] = -1j, 1j
    l[7] = np.diag([1, 1, -2]) / math.sqrt(3)
    return l / 2



# ---------------------------------------------------------------- brute force: explicit colour, no diagram list
def explicit_colour_me_hel(n, p, hel):
    """sum over all external colours of |M|^2 for one helicity configuration, by a colour-dressed off-shell
    recursion with explicit f^{abc}, T^a_{ij} and 4x4 gamma matrices; external states from their defining
    eigenvalue equations (def_u, def_v, def_eps).  No diagram enumeration, no colour-flow basis."""
    T = gell_mann()
    f = np.zeros((8, 8, 8), complex)
    for a in range(8):
        for b in range(8):
            comm = T[a] @ T[b] - T[b] @ T[a]
            for c in range(8):
                f[a, b, c] = -2j * np.trace(comm @ T[c])
    mt = PRM["mt"]
    part = lambda g: g if g < 2 else g + 2
    full = (1 << n) - 1
    K = {m: sum((1 if g < 2 else -1) * p[part(g)] for g in range(n) if m >> g & 1) for m in range(1, full + 1)}
    K[0] = np.zeros(4)
    L = "ABCDEFGH"                                                # einsum letter of each gluon's external colour
    letters = lambda m: "".join(L[g] for g in range(n) if m >> g & 1)
    low = lambda V: np.tensordot(METRIC, V, axes=(1, 0))
    G = {}
    masks = sorted(range(1, full + 1), key=lambda m: (bin(m).count("1"), m))
    for m in masks:
        bits = [g for g in range(n) if m >> g & 1]
        if len(bits) == 1:
            g = bits[0]
            e = def_eps(p[part(g)], hel[part(g)])
            e = e if g < 2 else e.conj()
            G[m] = np.einsum("m,ca->mca", e, np.eye(8))          # [mu, open colour, external colour]
            continue
        acc = 0
        lowbit = m & -m
        subs = [A for A in range(1, m) if (A & m) == A]
        for A in subs:                                           # three-gluon vertex
            B = m ^ A
            if not A & lowbit:
                continue
            k1, k2 = K[A], K[B]
            k3 = -(k1 + k2)
            V1, V2 = G[A], G[B]
            la, lb, ls = letters(A), letters(B), letters(m)
            t1 = np.einsum(f"ma{la},mb{lb},r->rab{la}{lb}", low(V1), V2, k1 - k2)
            t2 = np.einsum(f"m,ma{la},rb{lb}->rab{la}{lb}", METRIC @ (k2 - k3), V1, V2)
            t3 = np.einsum(f"m,mb{lb},ra{la}->rab{la}{lb}", METRIC @ (k3 - k1), V2, V1)
            acc = acc + GS * np.einsum(f"abc,rab{la}{lb}->rc{ls}", f, t1 + t2 + t3)
        for A in subs:                                           # four-gluon vertex
            if not A & lowbit:
                continue
            rest = m ^ A
            lowr = rest & -rest
            for B in [x for x in range(1, rest) if (x & rest) == x and x & lowr]:
                Cc = rest ^ B
                V1, V2, V3 = G[A], G[B], G[Cc]
                la, lb, lc, ls = letters(A), letters(B), letters(Cc), letters(m)
                tot = 0
                for fa, fb, kin in (("abe", "cde", (("13", 2, +1), ("23", 1, -1))),
                                    ("ace", "bde", (("12", 3, +1), ("23", 1, -1))),
                                    ("ade", "bce", (("12", 3, +1), ("13", 2, -1)))):
                    for pair, free, sign in kin:
                        idx = {1: f"a{la}", 2: f"b{lb}", 3: f"c{lc}"}
                        Vs = {1: V1, 2: V2, 3: V3}
                        i, j = int(pair[0]), int(pair[1])
                        tot = tot + sign * np.einsum(f"{fa},{fb},m{idx[i]},m{idx[j]},s{idx[free]}->sd{ls}",
                                                     f, f, low(Vs[i]), Vs[j], Vs[free], optimize=True)
                acc = acc + (-1j * GS ** 2) * tot
        k2 = K[m] @ METRIC @ K[m]
        G[m] = (-1j / k2) * acc
    # quark line from the outgoing t: Psi[S][spinor, i, j, colours]
    pt, ptb = p[2], p[3]
    ub = def_u(pt, mt, hel[2]).conj() @ GAM[0]
    v = def_v(ptb, mt, hel[3])
    Psi = {0: np.einsum("b,ij->bij", ub, np.eye(3))}
    for m in masks:
        if m == full:
            continue
        q = pt - K[m]
        prop = 1j * (slash(q) + mt * I4) / (q @ METRIC @ q - mt ** 2)
        acc = 0
        for A in [x for x in range(1, m + 1) if (x & m) == x]:
            S = m ^ A
            ls, la, lm = letters(S), letters(A), letters(m)
            acc = acc + np.einsum(f"bij{ls},mbe,mc{la},cjk,ea->aik{lm}", Psi[S], GAM, low(G[A]), T, prop, optimize=True) * (1j * GS)
        Psi[m] = acc
    M = 0
    for A in [x for x in range(1, full + 1)]:
        S = full ^ A
        ls, la, lm = letters(S), letters(A), letters(full)
        M = M + np.einsum(f"bij{ls},mbe,mc{la},cjk,e->ik{lm}", Psi[S], GAM, low(G[A]), T, v, optimize=True) * (1j * GS)
    return float((abs(M) ** 2).sum())
