"""Pins for the oracle's Philox4x32-10 and uniform conversion (O5)."""
import os

import numpy as np

HERE = os.path.dirname(__file__)


def test_known_answers(olib):
    n = 0
    for line in open(os.path.join(HERE, "golden", "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        out = olib.philox(w[0:4], w[4:6])
        assert [int(v) for v in out] == w[6:10]
        n += 1
    assert n == 3


def test_uniform_conversion_and_layout(olib):
    # block n of a stream yields ((x0<<32|x1)>>11) 2^-53 and the same for (x2,x3); key = (seed_lo ^ tag, seed_hi)
    seed, tag = 0x123456789ABCDEF0, 0x454D4954
    u = olib.stream(seed, tag, 5, 6, 7, 6)
    for blk in range(3):
        o = olib.philox([5, 6, 7, blk], [(seed & 0xFFFFFFFF) ^ tag, seed >> 32])
        a = ((int(o[0]) << 32 | int(o[1])) >> 11) * 2.0 ** -53
        b = ((int(o[2]) << 32 | int(o[3])) >> 11) * 2.0 ** -53
        assert u[2 * blk] == a and u[2 * blk + 1] == b
    assert np.all((u >= 0) & (u < 1))


def test_uniformity_chi2(olib):
    n = 2_000_000
    u = olib.stream(1, 0x53544550, 11, 0, 0, n)
    h, _ = np.histogram(u, bins=256, range=(0, 1))
    chi2 = np.sum((h - n / 256) ** 2 / (n / 256))
    assert 170 < chi2 < 350          # 255 dof: mean 255, sigma 22.6
    assert abs(u.mean() - 0.5) < 4 * (1 / 12 / n) ** 0.5
    # lag-1 correlation
    c = np.corrcoef(u[:-1], u[1:])[0, 1]
    assert abs(c) < 4 / n ** 0.5
