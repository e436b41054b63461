"""Pins for the oracle's cross-section sums and hit-or-miss unweighting (include/me.h me_unweight):
the unweighted e+ e- -> mu+ mu- sample must reproduce the closed-form forward-backward asymmetry, the acceptance
must equal mean/max, and the sums the closed-form cross section."""
import math

import numpy as np

PRM = dict(mz=91.188, wz=2.441404, aewm1=132.507, sw2=0.2222)
SIGMA_EPEM = 1.21298820395e-10       # GeV^-2, SURVEY.md §8(c)


def afb_closed_form(s):
    sw2 = PRM["sw2"]; sw = math.sqrt(sw2); cw = math.sqrt(1 - sw2)
    gL, gR = (-0.5 + sw2) / (sw * cw), sw2 / (sw * cw)
    A = lambda ga, gb: 1 + ga * gb * s / complex(s - PRM["mz"] ** 2, PRM["mz"] * PRM["wz"])
    a = abs(A(gL, gL)) ** 2 + abs(A(gR, gR)) ** 2
    b = abs(A(gL, gR)) ** 2 + abs(A(gR, gL)) ** 2
    return (a - b) / (2 * (a + b))       # <cos theta> for d sigma/dc ~ a (1+c)^2 + b (1-c)^2


def test_unweighted_sample_reproduces_closed_form_asymmetry_and_cross_section(orc):
    n, sqs = 60000, 1500.0
    p, w = orc.events(0, n, seed=20230331)
    me = orc.me(0, p)
    s1, s2, wmax, acc = orc.unweight(w, me, 1.0 / (2 * sqs * sqs), seed=99)
    sigma, err = s1 / n, math.sqrt((s2 / n - (s1 / n) ** 2) / n)
    assert abs(sigma - SIGMA_EPEM) < 4 * err
    # acceptance = mean / max (hit-or-miss), within its binomial error
    eff = s1 / (n * wmax)
    assert abs(acc.mean() - eff) < 5 * math.sqrt(eff * (1 - eff) / n)
    # c = cos(angle between e- (particle 1, along -z) and mu- (particle 3))
    c = -p[:, 3, 3] / np.linalg.norm(p[:, 3, 1:], axis=1)
    ca = c[acc]
    target = afb_closed_form(sqs * sqs)
    assert abs(ca.mean() - target) < 4 * ca.std() / math.sqrt(ca.size)
    assert abs(target) > 0.05                                  # the pin has teeth: flat acceptance would give 0
    # a fixed wmax above the batch maximum lowers the acceptance in proportion
    _, _, _, acc2 = orc.unweight(w, me, 1.0 / (2 * sqs * sqs), seed=99, wmax=2 * wmax)
    assert abs(acc2.mean() - eff / 2) < 5 * math.sqrt(eff / 2 / n)
    assert (acc2 <= acc).all()                                 # same uniforms: a subset


def test_unweighting_uniforms_are_the_stated_philox_words(orc):
    """u_i = u53(w0, w1) of Philox4x32-10 at counter (event lo, event hi, 'UNWT', 0): recomputed here word by word from the
    known-answer-tested block function; a rejected event has u * wmax >= w, an accepted one u * wmax < w."""
    n, seed, first = 300, 0x1234567890, (1 << 32) - 100            # crosses the 32-bit boundary of the event counter
    rng = np.random.default_rng(1)
    w, me = rng.uniform(0.5, 1.5, n), rng.uniform(0.0, 1.0, n)
    s1, s2, wmax, acc = orc.unweight(w, me, 2.0, seed=seed, first_event=first)
    ww = 2.0 * w * me
    assert wmax == ww.max() and abs(s1 - ww.sum()) < 1e-12 * s1 and abs(s2 - (ww * ww).sum()) < 1e-12 * s2
    for i in range(n):
        ev = first + i
        wd = orc.philox4x32_10([ev & 0xFFFFFFFF, ev >> 32, 0x554E5754, 0], [seed & 0xFFFFFFFF, seed >> 32])
        u = ((wd[0] >> 5) * 67108864.0 + (wd[1] >> 6) + 0.5) / 9007199254740992.0
        assert bool(acc[i]) == (u * wmax < ww[i])
