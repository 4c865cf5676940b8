"""Pins for the oracle's noise: Philox4x32-10 (O1) and uniform->normal (O2).  CPU only."""
import os

import numpy as np
import scipy.stats

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers(oracle):
    n = 0
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        out = oracle.philox4x32_10(w[0:4], w[4:6])
        assert [int(x) for x in out] == w[6:10]
        n += 1
    assert n == 3


def test_philox_is_a_bijection_on_small_counter_set(oracle):
    # distinct counters under one key give distinct blocks (Philox is a keyed permutation)
    seen = set()
    for c in range(2000):
        seen.add(tuple(int(x) for x in oracle.philox4x32_10([c, 0, 0, 0], [7, 9])))
    assert len(seen) == 2000


def test_normals_counter_layout(oracle):
    """component j of the noise for (p,q,t,stream) comes from counter (p,q,t,stream<<16 | j//4),
    word j%4 (reading R3): rebuild from the KAT-pinned block function + numpy Box-Muller."""
    seed = 0x0123456789ABCDEF
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for (p, q, t, stream, n) in [(0, 0, 0, 1, 4), (5, 17, 3, 2, 10), (1000000, 4095, 29, 3, 33)]:
        z = oracle.normals(seed, p, q, t, stream, n)
        for blk in range((n + 3) // 4):
            x = oracle.philox4x32_10([p, q, t, (stream << 16) | blk], key)
            u = (x.astype(np.float64) * 2.0 ** -32 + 2.0 ** -33)
            r0, r1 = np.sqrt(-2 * np.log(u[0])), np.sqrt(-2 * np.log(u[2]))
            ref = [r0 * np.cos(2 * np.pi * u[1]), r0 * np.sin(2 * np.pi * u[1]),
                   r1 * np.cos(2 * np.pi * u[3]), r1 * np.sin(2 * np.pi * u[3])]
            for j in range(4):
                if 4 * blk + j < n:
                    # fp32 libm vs fp64 numpy: the angle 2*pi*u is rounded to fp32 (<= 4e-7 abs)
                    assert abs(z[4 * blk + j] - ref[j]) < 5e-6 * max(1.0, abs(ref[j])) + 5e-6


def test_normals_streams_and_indices_differ(oracle):
    base = oracle.normals(1, 2, 3, 4, 1, 8)
    for args in [(1, 2, 3, 4, 2), (1, 3, 3, 4, 1), (1, 2, 4, 4, 1), (1, 2, 3, 5, 1), (2, 2, 3, 4, 1)]:
        other = oracle.normals(args[0], args[1], args[2], args[3], args[4], 8)
        assert not np.allclose(base, other)
    # prefix property: asking for fewer components returns the same leading ones
    assert np.array_equal(oracle.normals(1, 2, 3, 4, 1, 5), base[:5])


def test_normals_moments(oracle):
    z = np.concatenate([oracle.normals(42, p, 0, 0, 1, 1000) for p in range(1000)]).astype(np.float64)
    assert z.size == 10 ** 6
    assert abs(z.mean()) < 4e-3
    assert abs(z.var() - 1.0) < 6e-3
    assert abs(scipy.stats.kurtosis(z, fisher=False) - 3.0) < 0.02
    assert abs(scipy.stats.skew(z)) < 0.01
    assert np.abs(z).max() <= 6.8          # u >= 2^-33  =>  r <= sqrt(2*33*ln2) = 6.76
    # library check of the whole law: Kolmogorov-Smirnov against N(0,1)
    assert scipy.stats.kstest(z[:200000], "norm").pvalue > 1e-3
    # components are uncorrelated across the 4 words of a block
    zz = z.reshape(-1, 4)
    c = np.corrcoef(zz.T)
    assert np.abs(c - np.eye(4)).max() < 0.01


def test_resample_word_is_stream4_word0(oracle):
    seed = 987654321987
    x = oracle.philox4x32_10([0, 0, 0, 4 << 16], [seed & 0xFFFFFFFF, seed >> 32])
    assert oracle.resample_word(seed) == int(x[0])
