"""Pins for the oracle's event-by-event helicity / leading-colour choice (rule in include/me.h
me_select_helicity_color): an independent numpy inverse CDF (cumsum + searchsorted) driven by the pinned Philox, the
sampling frequencies against the exact probabilities (chi-square), and the mask."""
import numpy as np
import pytest

TAG = 0x53454C45


def uniforms(orc, seed, ev):
    w = orc.philox4x32_10([ev & 0xFFFFFFFF, ev >> 32, TAG, 0], [seed & 0xFFFFFFFF, seed >> 32])
    u = lambda a, b: ((a >> 5) * 67108864.0 + (b >> 6) + 0.5) / 9007199254740992.0
    return u(w[0], w[1]), u(w[2], w[3])


@pytest.mark.parametrize("proc,mask", [(0, 0x0660), (1, 0x9FF9), (2, (1 << 32) - 1), (3, (1 << 64) - 1)])
def test_selection_is_the_inverse_cdf_of_the_stated_weights(orc, proc, mask):
    n, seed, first = (60, 11, 5) if proc == 3 else (200, 11, 5)
    p, _ = orc.events(proc, n, seed=77)
    ihel, icol = orc.select(proc, p, seed, first, mask)
    _, mh = orc.me(proc, p, per_helicity=True)
    good = np.array([(mask >> h) & 1 for h in range(mh.shape[1])], dtype=float)
    for e in range(n):
        u1, u2 = uniforms(orc, seed, first + e)
        w = mh[e] * good
        cum = np.cumsum(w)
        k = int(np.searchsorted(cum, u1 * cum[-1], side="left"))
        while w[k] == 0:                                   # boundaries sit on positive weights only
            k += 1
        assert ihel[e] == k
        assert (mask >> k) & 1
        if proc == 0:
            assert icol[e] == 0
        else:
            j = orc.jamps(proc, p[e], k)
            cj = np.cumsum(np.abs(j) ** 2)
            assert icol[e] == int(np.searchsorted(cj, u2 * cj[-1], side="left"))


def test_selection_frequencies_follow_the_probabilities(orc):
    """one gg -> tt~g phase-space point replicated over 40000 event counters: chi-square of helicity and colour counts"""
    proc, n = 2, 40000
    p1, _ = orc.events(proc, 1, seed=5)
    p = np.repeat(p1, n, axis=0)
    ihel, icol = orc.select(proc, p, 123456789, 0, (1 << 32) - 1)
    _, mh = orc.me(proc, p1, per_helicity=True)
    ph = mh[0] / mh[0].sum()
    counts = np.bincount(ihel, minlength=32)
    sel = ph * n > 5
    chi2 = ((counts[sel] - ph[sel] * n) ** 2 / (ph[sel] * n)).sum()
    assert chi2 < sel.sum() + 5 * np.sqrt(2 * sel.sum())          # within ~5 sigma of the chi-square mean
    pc = np.zeros(6)
    for h in range(32):
        j = np.abs(orc.jamps(proc, p1[0], h)) ** 2
        pc += ph[h] * j / j.sum()
    cc = np.bincount(icol, minlength=6)
    chi2c = ((cc - pc * n) ** 2 / (pc * n)).sum()
    assert chi2c < 6 + 5 * np.sqrt(12)


def test_selection_respects_the_mask(orc):
    p, _ = orc.events(1, 50, seed=3)
    ihel, _ = orc.select(1, p, 1, 0, 1 << 6)
    assert (ihel == 6).all()
