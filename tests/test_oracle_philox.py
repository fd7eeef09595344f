"""P14: the oracle's Philox4x32-10 against published known-answer vectors and uniformity (CPU only)."""
import os

import numpy as np

from oracle import philox

HERE = os.path.dirname(os.path.abspath(__file__))


def test_philox_known_answer_vectors():
    n = 0
    for line in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.replace("->", " ").split()]
        out = philox.philox4x32_10(w[0], w[1], w[2], w[3], w[4], w[5])
        assert [int(o) for o in out] == w[6:10]
        n += 1
    assert n == 3


def test_philox_is_a_bijection_of_the_counter_and_depends_on_every_input():
    base = [int(o) for o in philox.philox4x32_10(1, 2, 3, 4, 5, 6)]
    for pos in range(6):
        args = [1, 2, 3, 4, 5, 6]
        args[pos] += 1
        assert [int(o) for o in philox.philox4x32_10(*args)] != base
    c0 = np.arange(4096)
    outs = philox.philox4x32_10(c0, 0, 0, 0, 7, 9)
    assert len({tuple(int(o[i]) for o in outs) for i in range(4096)}) == 4096


def test_uniform_maps():
    x = np.array([0, 0x1FF, 0x200, 0xFFFFFFFF], dtype=np.uint32)
    r = philox.uniform_pm1(x)
    assert r[0] == r[1] == -1.0 + 2.0 ** -23 and r[3] == 1.0 - 2.0 ** -23
    assert np.all(r.astype(np.float32).astype(np.float64) == r)          # exact in fp32 (S11)
    u = philox.uniform_01(x)
    assert u[0] == 2.0 ** -24 and u[3] == 1.0 - 2.0 ** -24
    x0, x1 = philox.site_words(1 << 18, 3, 0, 12345)
    r0, r1 = philox.uniform_pm1(x0), philox.uniform_pm1(x1)
    n = r0.size
    assert abs(r0.mean()) < 5 / np.sqrt(3 * n) and abs(r1.mean()) < 5 / np.sqrt(3 * n)
    assert abs((r0 ** 2).mean() - 1 / 3) < 5 * np.sqrt(4 / 45 / n)      # var of r^2 = 1/5 - 1/9
    assert abs((r0 * r1).mean()) < 5 / 3 / np.sqrt(n)
    assert abs(np.corrcoef(r0[:-1], r0[1:])[0, 1]) < 5 / np.sqrt(n)


def test_streams_and_steps_are_independent_counters():
    a = philox.site_words(64, 0, 0, 1)
    b = philox.site_words(64, 1, 0, 1)
    c = philox.site_words(64, 0, 1, 1)
    d = philox.site_words(64, 0, 0, 2)
    for other in (b, c, d):
        assert not np.array_equal(a[0], other[0])
    # 64-bit site index: the high word goes to counter word 1
    hi = philox.philox4x32_10(5, 1, 0, 0, 1, 0)
    lo = philox.philox4x32_10(5, 0, 0, 0, 1, 0)
    assert int(hi[0]) != int(lo[0])
