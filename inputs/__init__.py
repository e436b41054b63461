"""Seeded-input descriptions shared by tests, bench and smoke — NO method arithmetic here.

Holds only (a) the BASELINE.json config table (process, events, seed, sqrt_s, SM parameters) and
(b) pure layout transforms between AoS [n][npar][4] and the library's AoSoA
[ceil(n/P)][npar][4][P] momentum layout (include/me.h).  Philox and RAMBO are part of the method
(SURVEY §8(a) a0,a1) and are implemented twice, independently: oracle/ (host) and the CUDA library.
"""
import numpy as np

# (mz, wz, aewm1, sw2, mt, wt, alpha_s) — BASELINE.json configs
SM_PARAMS = (91.188, 2.441404, 132.507, 0.2222, 173.0, 0.0, 0.118)
SQRT_S = 1500.0

# cfg index (0-based) -> description; 'process' is the me_process enum value of include/me.h
CONFIGS = [
    dict(name="epem_mupmum", label="e+ e- -> mu+ mu-", process=0, npar=4, nfinal=2, events=16384, seed=20230331,
         precisions=("fp64",)),
    dict(name="gg_ttx", label="g g -> t t~", process=1, npar=4, nfinal=2, events=524288, seed=1,
         precisions=("fp64", "fp32")),
    dict(name="gg_ttxg", label="g g -> t t~ g", process=2, npar=5, nfinal=3, events=1048576, seed=2,
         precisions=("fp64", "mixed", "fp32")),
    dict(name="gg_ttxgg", label="g g -> t t~ g g", process=3, npar=6, nfinal=4, events=524288, seed=3,
         precisions=("fp64", "mixed", "fp32")),
    dict(name="gg_ttxggg", label="g g -> t t~ g g g", process=4, npar=7, nfinal=5, events=65536, seed=4,
         precisions=("fp64", "mixed", "fp32")),
]


def final_masses(process, params=SM_PARAMS):
    mt = params[4]
    return {0: [0.0, 0.0], 1: [mt, mt], 2: [mt, mt, 0.0], 3: [mt, mt, 0.0, 0.0], 4: [mt, mt, 0.0, 0.0, 0.0]}[process]


def aos_to_aosoa(p, page):
    """[n][npar][4] -> flat AoSoA [ceil(n/page)][npar][4][page]; the tail page is padded by repeating the last event."""
    n, npar, _ = p.shape
    npages = (n + page - 1) // page
    pad = npages * page - n
    if pad:
        p = np.concatenate([p, np.repeat(p[-1:], pad, axis=0)], axis=0)
    return np.ascontiguousarray(p.reshape(npages, page, npar, 4).transpose(0, 2, 3, 1)).reshape(-1)


def aosoa_to_aos(flat, n, npar, page):
    npages = (n + page - 1) // page
    a = np.asarray(flat).reshape(npages, npar, 4, page).transpose(0, 3, 1, 2).reshape(npages * page, npar, 4)
    return np.ascontiguousarray(a[:n])
