"""ORACLE — TEST INFRASTRUCTURE ONLY (see me_oracle.cpp header).

ctypes wrappers around the scalar CPU oracle.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package; the product
package paper_2303_18244_b200 never does, and this package never imports it.

Momenta here are AoS numpy arrays [n][npar][4] (E,px,py,pz), float64.
"""
import ctypes
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_DIR, "liboracle.so")
_SRC = os.path.join(_DIR, "me_oracle.cpp")
_lib = None

# process ids (same numbering as SURVEY §8 cfg 1..5, zero based)
EPEM_MUPMUM, GG_TTX, GG_TTXG, GG_TTXGG, GG_TTXGGG = range(5)

# BASELINE.json configs: SM parameters (mz, wz, aewm1, sw2, mt, wt, alpha_s)
DEFAULT_PARAMS = (91.188, 2.441404, 132.507, 0.2222, 173.0, 0.0, 0.118)


def build(force=False):
    """Compile liboracle.so with g++ (-O2, OpenMP).  Building the checker is not using it."""
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(_SRC):
        return _SO
    cmd = ["g++", "-O2", "-std=c++17", "-fcx-limited-range", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC]
    subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.orc_me.restype = ctypes.c_int
        _lib.orc_rambo.restype = ctypes.c_int
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def info(process):
    out = (ctypes.c_int * 9)()
    if lib().orc_info(int(process), out):
        raise ValueError("bad process")
    keys = ("npar", "nglu", "ncomb", "avg_denom", "ncol", "ndiagrams", "n_gterms", "n_qterms", "n_closures")
    return dict(zip(keys, list(out)))


def count_gluon_subtrees(n):
    return lib().orc_count_gluon_subtrees(int(n))


def color_matrix(process):
    nc = info(process)["ncol"]
    out = np.zeros((nc, nc))
    if lib().orc_color_matrix(int(process), _dp(out)):
        raise ValueError("bad process")
    return out


def max_threads():
    return lib().orc_max_threads()


def me(process, p, params=DEFAULT_PARAMS, long_double=False, ward_leg=-1, per_helicity=False, nthreads=0):
    """|M|^2 averaged (all helicities summed, /avg_denom).  Returns me[n] (and me_hel[n][ncomb], not averaged)."""
    p = np.ascontiguousarray(p, dtype=np.float64)
    inf = info(process)
    assert p.ndim == 3 and p.shape[1] == inf["npar"] and p.shape[2] == 4
    n = p.shape[0]
    prm = np.asarray(params, dtype=np.float64)
    out = np.zeros(n)
    mh = np.zeros((n, inf["ncomb"])) if per_helicity else None
    rc = lib().orc_me(int(process), _dp(prm), _dp(p), ctypes.c_long(n), int(long_double), int(ward_leg),
                      _dp(out), _dp(mh) if per_helicity else None, int(nthreads))
    if rc:
        raise ValueError("orc_me failed")
    return (out, mh) if per_helicity else out


def helicity_mask(me_hel, threshold=1e-12):
    """h is good iff max over the filter events of ME_h/sum_h' ME_h' > threshold.  Returns int bit mask."""
    frac = me_hel / me_hel.sum(axis=1, keepdims=True)
    good = frac.max(axis=0) > threshold
    mask = 0
    for h, g in enumerate(good):
        if g:
            mask |= 1 << h
    return mask


def select(process, p, seed, first_event, mask, params=DEFAULT_PARAMS):
    """helicity / leading-colour choice per event (me_oracle.cpp orc_select) -> (ihel[n], icol[n]) int32"""
    p = np.ascontiguousarray(p, dtype=np.float64)
    n = p.shape[0]
    prm = np.asarray(params, dtype=np.float64)
    m = (ctypes.c_uint64 * 2)(mask & ((1 << 64) - 1), mask >> 64)
    ihel = np.zeros(n, dtype=np.int32); icol = np.zeros(n, dtype=np.int32)
    rc = lib().orc_select(int(process), _dp(prm), _dp(p), ctypes.c_long(n), ctypes.c_uint64(seed), ctypes.c_uint64(first_event), m,
                          ihel.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), icol.ctypes.data_as(ctypes.POINTER(ctypes.c_int)))
    if rc:
        raise ValueError("orc_select failed")
    return ihel, icol


def unweight(weight, me_values, flux, seed, first_event=0, wmax=0.0):
    """Cross-section sums and hit-or-miss unweighting, the plain definition (include/me.h me_unweight):
    w = flux * W * ME; returns (sum w, sum w^2, max w, accept[n] bool) with accept_i = u_i * wmax < w_i."""
    import math
    w = flux * np.asarray(weight, dtype=np.float64) * np.asarray(me_values, dtype=np.float64)
    n = w.shape[0]
    u = np.zeros(n)
    lib().orc_tagged_uniform(ctypes.c_uint64(seed), ctypes.c_uint64(first_event), ctypes.c_long(n), ctypes.c_uint32(0x554E5754), _dp(u))
    wm = float(w.max()) if wmax <= 0 else float(wmax)
    return math.fsum(w), math.fsum(w * w), float(w.max()), (u * wm < w)


def jamps(process, p_event, ihel, params=DEFAULT_PARAMS):
    p_event = np.ascontiguousarray(p_event, dtype=np.float64)
    nc = info(process)["ncol"]
    out = np.zeros((nc, 2))
    prm = np.asarray(params, dtype=np.float64)
    if lib().orc_jamps(int(process), _dp(prm), _dp(p_event), int(ihel), _dp(out)):
        raise ValueError("orc_jamps failed")
    return out[:, 0] + 1j * out[:, 1]


def external(kind, p, m, lam):
    """kind: 'u', 'v' or 'eps' -> 4 complex components."""
    k = {"u": 0, "v": 1, "eps": 2}[kind]
    p = np.ascontiguousarray(p, dtype=np.float64)
    out = np.zeros((4, 2))
    lib().orc_external(k, _dp(p), ctypes.c_double(m), int(lam), _dp(out))
    return out[:, 0] + 1j * out[:, 1]


def philox4x32_10(ctr, key):
    c = (ctypes.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (ctypes.c_uint32 * 2)(*[int(x) for x in key])
    o = (ctypes.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def philox_uniform(seed, first_event, n, per_event):
    out = np.zeros((n, per_event, 4))
    lib().orc_philox_uniform(ctypes.c_uint64(seed), ctypes.c_uint64(first_event), ctypes.c_long(n), int(per_event), _dp(out))
    return out


def rambo(masses, sqrt_s, rnd, long_double=False):
    """rnd[n][nfinal][4] -> (p[n][2+nfinal][4], weight[n])"""
    rnd = np.ascontiguousarray(rnd, dtype=np.float64)
    n, nf = rnd.shape[0], rnd.shape[1]
    m = np.asarray(masses, dtype=np.float64)
    assert m.shape[0] == nf
    p = np.zeros((n, nf + 2, 4))
    w = np.zeros(n)
    if lib().orc_rambo(int(nf), _dp(m), ctypes.c_double(sqrt_s), _dp(rnd), ctypes.c_long(n), _dp(p), _dp(w), int(long_double)):
        raise ValueError("orc_rambo failed")
    return p, w


# final-state masses per process (GeV), BASELINE.json configs
def final_masses(process, params=DEFAULT_PARAMS):
    mt = params[4]
    return {0: [0.0, 0.0], 1: [mt, mt], 2: [mt, mt, 0.0], 3: [mt, mt, 0.0, 0.0], 4: [mt, mt, 0.0, 0.0, 0.0]}[process]


def events(process, n, seed, sqrt_s=1500.0, first_event=0, params=DEFAULT_PARAMS):
    """Seeded RAMBO events exactly as BASELINE.json configs describe them (oracle-side Philox + RAMBO)."""
    masses = final_masses(process, params)
    rnd = philox_uniform(seed, first_event, n, len(masses))
    return rambo(masses, sqrt_s, rnd)
