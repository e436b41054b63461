"""The parity bar between the CUDA path and the oracle, in one place (used by tests/test_gpu_parity.py and by
tests/full_parity_report.py, which writes the all-events report kept under profiles/).

BASELINE.json north_star: relative |M|^2 error <= 1e-11 in FP64 and <= 1e-4 in FP32 / mixed, per event, against the oracle on
the same seeded events.  The FP64 reference is the oracle in long double.  SURVEY.md section 8(c) risk R1 (lines 381-394):
without cuts a few RAMBO points per 10^5 have a tiny invariant s_ij, gauge cancellations then amplify rounding in ANY binary64
evaluation, and such events "must be attributed, not hidden": an event is judged against

    tol_i = max(1e-11, 10 x |oracle_double_i / oracle_long_double_i - 1|)

i.e. against ten times the discrepancy the oracle itself shows between its two precisions on that event; 1e-11
stays the headline criterion and every event above it is listed with s_min/s and the oracle's own spread.  No arithmetic of the
method lives here: only comparisons of finished numbers.
"""
import numpy as np

TOL64, TOL32 = 1e-11, 1e-4
SPREAD_FACTOR = 10.0


def smin_over_s(p, sqrt_s=1500.0):
    """smallest |2 p_i.p_j| over parton pairs (the t t~ pair excluded: it is never a propagator by itself), over s"""
    npar = p.shape[1]
    d = lambda a, b: a[:, 0] * b[:, 0] - (a[:, 1:] * b[:, 1:]).sum(1)
    out = np.full(p.shape[0], np.inf)
    for i in range(npar):
        for j in range(i + 1, npar):
            if (i, j) == (2, 3):
                continue
            out = np.minimum(out, np.abs(2 * d(p[:, i], p[:, j])))
    return out / (sqrt_s ** 2)


def judge_fp64(out, ref_ld, ref_d):
    """-> dict: rel (per event), spread (oracle double vs long double), tol, above (indices with rel > 1e-11), failed (indices with
    rel > tol_i), oracle_above (events where the oracle's own spread exceeds 1e-11)"""
    rel = np.abs(out / ref_ld - 1)
    spread = np.abs(ref_d / ref_ld - 1)
    tol = np.maximum(TOL64, SPREAD_FACTOR * spread)
    return dict(rel=rel, spread=spread, tol=tol, above=np.nonzero(rel > TOL64)[0], failed=np.nonzero(~(rel <= tol))[0],
                oracle_above=np.nonzero(spread > TOL64)[0])


def judge_fp32(out, ref_ld):
    rel = np.abs(out / ref_ld - 1)
    return dict(rel=rel, above=np.nonzero(~(rel <= TOL32))[0], mean_ratio=float(out.mean() / ref_ld.mean() - 1))


def summary(rel):
    return dict(max=float(rel.max()), p999=float(np.quantile(rel, 0.999)), median=float(np.median(rel)))
