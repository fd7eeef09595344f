"""Philox4x32-10 counter-based generator, plain numpy (uint64 arithmetic on uint32 words).

ORACLE / TEST INFRASTRUCTURE -- see oracle/__init__.py.

The paper only says the Langevin term is made of "random numbers uniformly distributed over
[-zeta_max, zeta_max]" for "every mesh point and time step" and names no generator;
BASELINE.json's north_star fixes "a counter-based Philox noise generator" (reading S11).
The algorithm restated here is Philox-4x32 with 10 rounds of Salmon, Moraes, Dror, Shaw,
"Parallel random numbers: as easy as 1, 2, 3" (SC'11), Sec. 3.3 / Table 2:

    one round on counter (c0,c1,c2,c3) with key (k0,k1):
        (hi0, lo0) = mulhilo32(M0, c0);   (hi1, lo1) = mulhilo32(M1, c2)
        (c0,c1,c2,c3) <- (hi1 ^ c1 ^ k0,  lo1,  hi0 ^ c3 ^ k1,  lo0)
    between rounds the key is bumped by the Weyl constants (k0 += W0, k1 += W1).

Pinned (tests/test_oracle_philox.py) against the known-answer vectors published with that paper's
reference distribution (tests/golden/philox4x32_10_kat.txt) and against uniformity moments.
"""
import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = np.uint64(0x9E3779B9)      # golden ratio
_W1 = np.uint64(0xBB67AE85)      # sqrt(3) - 1
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Vectorised over the counter words.  All inputs are integers / integer arrays in [0, 2^32).
    Returns four uint32 arrays (the four output words)."""
    c0, c1, c2, c3 = (np.asarray(c, dtype=np.uint64) & _MASK for c in (c0, c1, c2, c3))
    c0, c1, c2, c3 = np.broadcast_arrays(c0, c1, c2, c3)
    k0 = np.uint64(int(k0) & 0xFFFFFFFF)
    k1 = np.uint64(int(k1) & 0xFFFFFFFF)
    for rnd in range(10):
        if rnd > 0:
            k0 = (k0 + _W0) & _MASK
            k1 = (k1 + _W1) & _MASK
        p0 = _M0 * c0                      # 32x32 -> 64 bit products, exact in uint64
        p1 = _M1 * c2
        hi0, lo0 = p0 >> _S32, p0 & _MASK
        hi1, lo1 = p1 >> _S32, p1 & _MASK
        c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
    return tuple(c.astype(np.uint32) for c in (c0, c1, c2, c3))


def site_words(n_sites, step, stream, seed):
    """Words (x0, x1) for every global site index m = 0..n_sites-1 (reading S11):
    key = (seed_lo, seed_hi), counter = (m_lo, m_hi, step, stream); stream 0 = noise, 1 = init."""
    m = np.arange(n_sites, dtype=np.uint64)
    x0, x1, _, _ = philox4x32_10(m & _MASK, m >> _S32, step, stream,
                                 seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)
    return x0, x1


def uniform_pm1(x):
    """uint32 word -> uniform in (-1, 1): r = ((x >> 9) + 0.5) * 2^-22 - 1  (S11).
    23 random bits; every value is an odd multiple of 2^-23, so it is exact in fp32 and fp64 alike,
    symmetric about 0 and never +-1."""
    return ((x >> np.uint32(9)).astype(np.float64) + 0.5) * 2.0 ** -22 - 1.0


def uniform_01(x):
    """uint32 word -> uniform in (0, 1): ((x >> 9) + 0.5) * 2^-23  (S13, Box-Muller input)."""
    return ((x >> np.uint32(9)).astype(np.float64) + 0.5) * 2.0 ** -23
