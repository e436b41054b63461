"""Pins for the oracle's Philox4x32-10 and RAMBO (SURVEY §8(c) 'Pins', Q12, Q14)."""
import math

import numpy as np
import pytest
from scipy import integrate, stats

# Random123 known-answer vectors for philox4x32-10 (Salmon et al. SC'11 distribution, kat_vectors;
# also listed in SURVEY §8(c) Pins/Philox)
KAT = [
    ([0, 0, 0, 0], [0, 0], [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]),
    ([0xFFFFFFFF] * 4, [0xFFFFFFFF] * 2, [0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD]),
    ([0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344], [0xA4093822, 0x299F31D0],
     [0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1]),
]


@pytest.mark.parametrize("ctr,key,exp", KAT)
def test_philox_known_answers(orc, ctr, key, exp):
    assert orc.philox4x32_10(ctr, key) == exp


def test_philox_uniform_mapping_worked_examples(orc):
    # SURVEY Q14 worked example: key=(seed lo, seed hi), ctr=(event lo, event hi, particle, j)
    assert orc.philox4x32_10([0, 0, 0, 0], [3, 0]) == [0xD1104D77, 0x1DE847CE, 0xA7F2EC5A, 0xC3E627F9]
    assert orc.philox4x32_10([0, 0, 0, 1], [3, 0]) == [0x14E87FAE, 0x8C2DD169, 0x74FCB00C, 0xA4773893]
    u = orc.philox_uniform(3, 0, 1, 4)[0, 0]
    assert u.tolist() == [0.8166550034048079, 0.6560504642518659, 0.08167265018503461, 0.45698071004781254]
    u = orc.philox_uniform(3, 524287, 1, 4)[0, 3]
    assert u.tolist() == [0.952241511877556, 0.9315503744350817, 0.8785202801284302, 0.9327533510747661]


def test_philox_uniform_formula_from_words(orc):
    # u = ((w0>>5)*2^26 + (w1>>6) + 0.5) * 2^-53, strictly inside (0,1); windows are consistent
    w = orc.philox4x32_10([7, 0, 2, 0], [99, 1]) + orc.philox4x32_10([7, 0, 2, 1], [99, 1])
    u = orc.philox_uniform(99 + (1 << 32), 7, 1, 3)[0, 2]
    for i in range(4):
        exact = ((w[2 * i] >> 5) * 2 ** 26 + (w[2 * i + 1] >> 6) + 0.5) / 2 ** 53
        assert u[i] == exact
    big = orc.philox_uniform(5, 0, 2000, 3)
    assert big.min() > 0.0 and big.max() < 1.0
    assert np.array_equal(orc.philox_uniform(5, 100, 50, 3), big[100:150])
    assert abs(big.mean() - 0.5) < 4 / math.sqrt(12 * big.size)


def mass2(p):
    return p[..., 0] ** 2 - (p[..., 1:] ** 2).sum(-1)


@pytest.mark.parametrize("process", [0, 1, 2, 3, 4])
def test_rambo_momentum_conservation_and_mass_shell(orc, process):
    p, w = orc.events(process, 2000, seed=11 + process)
    masses = np.array(orc.final_masses(process))
    tot = p[:, 2:].sum(axis=1)
    # boost to the CM frame divides by M = sqrt(Q.Q): relative rounding grows like eps*(Q0/M)^2 for
    # nearly collinear q's, so the bound is 1e-11 on the worst event and 1e-13 on the median
    dev = np.abs(tot - np.array([1500.0, 0, 0, 0])).max(axis=1) / 1500
    assert dev.max() < 1e-11 and np.median(dev) < 1e-13
    dm2 = np.abs(mass2(p[:, 2:]) - masses ** 2)
    assert np.median(dm2) < 1e-9 and dm2.max() < 1e-11 * 1500 ** 2   # GeV^2; same conditioning remark
    # beams: C1
    assert np.array_equal(p[:, 0], np.tile([750.0, 0, 0, 750.0], (2000, 1)))
    assert np.array_equal(p[:, 1], np.tile([750.0, 0, 0, -750.0], (2000, 1)))
    assert (w > 0).all() and (p[:, 2:, 0] > 0).all()


def test_rambo_two_body_volume_closed_form(orc):
    rnd = orc.philox_uniform(1, 0, 100, 2)
    s = 1500.0 ** 2
    _, w0 = orc.rambo([0.0, 0.0], 1500.0, rnd)
    assert np.allclose(w0, 1 / (8 * math.pi), rtol=1e-14)
    _, wm = orc.rambo([173.0, 173.0], 1500.0, rnd)
    beta = math.sqrt(1 - 4 * 173.0 ** 2 / s)
    assert np.allclose(wm, beta / (8 * math.pi), rtol=1e-12)
    # unequal masses: |p*|/(4 pi sqrt s)
    _, wu = orc.rambo([173.0, 50.0], 1500.0, rnd)
    pst = math.sqrt((s - (173 + 50) ** 2) * (s - (173 - 50) ** 2)) / (2 * 1500)
    assert np.allclose(wu, pst / (4 * math.pi * 1500), rtol=1e-12)


def test_rambo_massless_volumes(orc):
    s = 1500.0 ** 2
    for n, vol in ((3, s / (256 * math.pi ** 3)), (4, s ** 2 / (24576 * math.pi ** 5))):
        _, w = orc.rambo([0.0] * n, 1500.0, orc.philox_uniform(2, 0, 10, n))
        assert np.allclose(w, vol, rtol=1e-13)


def test_rambo_three_body_massive_volume_vs_dalitz_integral(orc):
    # Phi_3 = 1/(128 pi^3 s) * Dalitz area;  MC mean of RAMBO weights estimates Phi_3
    m1, m2, m3, rs = 173.0, 173.0, 0.0, 1500.0
    s = rs * rs

    def lam(a, b, c):
        return a * a + b * b + c * c - 2 * a * b - 2 * a * c - 2 * b * c

    def width(m12sq):
        m12 = math.sqrt(m12sq)
        e2 = (m12sq - m1 ** 2 + m2 ** 2) / (2 * m12)
        e3 = (s - m12sq - m3 ** 2) / (2 * m12)
        return 4 * math.sqrt(max(e2 * e2 - m2 ** 2, 0.0)) * math.sqrt(max(e3 * e3 - m3 ** 2, 0.0))

    area, _ = integrate.quad(width, (m1 + m2) ** 2, (rs - m3) ** 2, epsabs=0, epsrel=1e-10)
    phi3 = area / (128 * math.pi ** 3 * s)
    n = 200000
    _, w = orc.rambo([m1, m2, m3], rs, orc.philox_uniform(77, 0, n, 3))
    est, err = w.mean(), w.std() / math.sqrt(n)
    assert abs(est - phi3) < 4 * err
    assert err / phi3 < 2e-3


def test_rambo_two_body_isotropy(orc):
    p, _ = orc.rambo([0.0, 0.0], 1500.0, orc.philox_uniform(5, 0, 20000, 2))
    cos = p[:, 2, 3] / 750.0
    phi = np.arctan2(p[:, 2, 2], p[:, 2, 1])
    assert stats.kstest(cos, stats.uniform(-1, 2).cdf).pvalue > 1e-3
    assert stats.kstest(phi, stats.uniform(-math.pi, 2 * math.pi).cdf).pvalue > 1e-3


def test_rambo_double_vs_long_double(orc):
    rnd = orc.philox_uniform(4, 0, 500, 5)
    m = orc.final_masses(4)
    p, w = orc.rambo(m, 1500.0, rnd)
    pl, wl = orc.rambo(m, 1500.0, rnd, long_double=True)
    assert np.abs(p - pl).max() < 1e-10 and np.abs(w / wl - 1).max() < 1e-12
