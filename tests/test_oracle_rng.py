"""Pins for the oracle's counter-based RNG (R10, R11)."""
import os

import numpy as np

import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers():
    n = 0
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert list(O.philox4x32_10(w[0:4], w[4:6])) == w[6:10]
        n += 1
    assert n == 3


def test_philox_counter_sensitivity():
    base = O.philox4x32_10([1, 2, 3, 4], [5, 6])
    for k in range(4):
        c = [1, 2, 3, 4]
        c[k] += 1
        assert not np.array_equal(O.philox4x32_10(c, [5, 6]), base)
    assert not np.array_equal(O.philox4x32_10([1, 2, 3, 4], [6, 6]), base)
    assert not np.array_equal(O.philox4x32_10([1, 2, 3, 4], [5, 7]), base)


def test_u01_range_symmetry_exactness():
    lo, hi = O.u01(0), O.u01(0xFFFFFFFF)
    assert lo == 2.0 ** -24 and hi == 1.0 - 2.0 ** -24
    for x in (0, 1, 511, 512, 0x7FFFFFFF, 0x80000000, 0xFFFFFE00, 0xFFFFFFFF, 123456789):
        u = O.u01(x)
        assert u == ((x >> 9) + 0.5) * 2.0 ** -23          # exactly representable in fp32
        assert O.u01(0xFFFFFFFF - x) == 1.0 - u            # symmetric about 1/2
        assert 0.0 < u < 1.0


def test_slot_uniforms_mapping():
    """even slot <- (x0,x1), odd slot <- (x2,x3) of counter (site, sweep, sample<<16 | slot>>1, domain)."""
    seed = 0x0123456789ABCDEF
    for (site, sweep, sample, slot, dom) in [(0, 0, 0, 0, 0), (7, 3, 2, 5, 1), (100000, 77, 31, 62, 1), (9, 1, 0, 63, 1)]:
        x = O.philox4x32_10([site, sweep, (sample << 16) | (slot >> 1), dom], [seed & 0xFFFFFFFF, seed >> 32])
        u1, u2 = O.slot_uniforms(seed, dom, site, sweep, sample, slot)
        k = 2 * (slot & 1)
        assert (u1, u2) == (O.u01(x[k]), O.u01(x[k + 1]))


def test_uniform_moments():
    us = np.array([O.slot_uniforms(42, 1, s, 1, 0, r) for s in range(2000) for r in range(4)])
    assert abs(us.mean() - 0.5) < 4 * np.sqrt(1 / 12 / us.size)
    assert abs(us.var() - 1 / 12) < 0.004
    assert abs(np.corrcoef(us[:, 0], us[:, 1])[0, 1]) < 0.05


def test_init_theta_uniform():
    th = O.init_theta(512, 8, 99, 3)
    assert th.dtype == np.float32 and th.min() > 0 and th.max() < 2 * np.pi + 1e-6
    u1, _ = O.slot_uniforms(99, 0, 17, 0, 3, 5)
    assert th[17, 5] == np.float32(np.float32(6.2831855) * np.float32(u1))
    h, _ = np.histogram(th, bins=16, range=(0, 2 * np.pi))
    exp = th.size / 16
    assert ((h - exp) ** 2 / exp).sum() < 45        # chi2, 15 dof
