"""Pins for the oracle's exact-integer systematic resampler (O7, reading R6) and the
normalised weights (O6).  CPU only.

What fixes the expected values here (none of it is the oracle's own code):
  * the count invariants of systematic resampling (north_star: counts lie in floor/ceil of N*w_i and
    sum to N),
  * special cases with a unique answer (uniform weights -> identity, one-hot -> all copies),
  * numpy.searchsorted on an exactly representable (dyadic) CDF (library special case),
  * brute force over every comb offset with python's unbounded integers / Fractions for N <= 4.
"""
from fractions import Fraction

import numpy as np
import pytest

X0S = [0, 1, 12345, 2 ** 31, 2 ** 32 - 1]


def _counts(anc, N):
    return np.bincount(anc, minlength=N)


def _quant(v):
    """q_i = floor(v_i * 2^32) with python integers (v_i is an fp32 in [0,1]: exact)."""
    return [int(Fraction(float(x)) * (1 << 32)) for x in v]


def test_counts_floor_ceil_and_sum(oracle):
    rng = np.random.default_rng(0)
    for N in (1, 2, 3, 17, 256, 1000, 4096, 65536):
        for trial in range(3):
            logw = 2.0 * rng.standard_normal(N)
            v = np.exp(logw - logw.max()).astype(np.float32)
            for x0 in X0S:
                anc, st = oracle.resample_systematic_x0(v, x0)
                assert st == 0
                assert anc.min() >= 0 and anc.max() < N
                assert np.all(np.diff(anc) >= 0)                  # non-decreasing
                cnt = _counts(anc, N)
                assert cnt.sum() == N
                q = np.array(_quant(v), dtype=object)
                W = int(q.sum())
                lo = np.array([(N * int(qi)) // W for qi in q])
                hi = np.array([-((-N * int(qi)) // W) for qi in q])
                assert np.all(cnt >= lo) and np.all(cnt <= hi)


def test_uniform_weights_give_identity(oracle):
    for N in (1, 2, 5, 64, 1000, 4097):
        for val in (1.0, 0.5, 0.3):          # any constant: only relative weights matter
            v = np.full(N, val, np.float32)
            for x0 in X0S:
                anc, st = oracle.resample_systematic_x0(v, x0)
                assert st == 0
                assert np.array_equal(anc, np.arange(N))


def test_one_hot_weight_gives_all_copies(oracle):
    for N in (1, 3, 100, 1025):
        for j in {0, N // 2, N - 1}:
            v = np.zeros(N, np.float32)
            v[j] = 1.0
            for x0 in X0S:
                anc, st = oracle.resample_systematic_x0(v, x0)
                assert st == 0
                assert np.all(anc == j)


def test_zero_weight_particles_never_chosen(oracle):
    rng = np.random.default_rng(3)
    N = 777
    v = rng.uniform(0, 1, N).astype(np.float32)
    dead = rng.uniform(size=N) < 0.6
    v[dead] = 0.0
    v[np.argmax(~dead)] = 1.0
    for x0 in X0S:
        anc, _ = oracle.resample_systematic_x0(v, x0)
        assert not np.any(dead[anc])


def test_all_zero_weights_flagged(oracle):
    anc, st = oracle.resample_systematic_x0(np.zeros(9, np.float32), 5)
    assert st == -2
    assert np.array_equal(anc, np.arange(9))
    # weights below 2^-32 of the maximum quantise to zero as well
    anc, st = oracle.resample_systematic_x0(np.full(9, 1e-12, np.float32), 5)
    assert st == -2


def test_dyadic_weights_match_numpy_searchsorted(oracle):
    """Multiples of 2^-10: the fp64 cumsum is exact, so the textbook
    searchsorted(cumsum(w)/sum, (k+u)/N, side='right') is exact too (library special case)."""
    rng = np.random.default_rng(11)
    for N in (8, 64, 1024, 4096):
        for trial in range(4):
            m = rng.integers(0, 1025, size=N)
            m[rng.integers(0, N)] = 1024
            v = (m / 1024.0).astype(np.float32)
            for x0 in [0, 2 ** 31, 3 << 29, 123 << 20]:     # x0 / 2^32 dyadic as well
                anc, st = oracle.resample_systematic_x0(v, x0)
                assert st == 0
                c = np.cumsum(m.astype(np.float64))             # integers < 2^53: exact
                W = c[-1]
                U = np.floor(x0 * W / 2.0 ** 32)                 # exact: W < 2^23, x0 has <= 12 bits
                pts = (np.arange(N) * W + U) / N                 # comb points in CDF units
                # exactness guard: N is a power of two so the division is exact
                ref = np.searchsorted(c, pts, side="right")
                assert np.array_equal(anc, ref)


def _brute(v, x0):
    """i_k = min{ i : C_i / W > (k + U/W) / N } with exact rationals, U = floor(x0 W / 2^32)."""
    q = _quant(v)
    N = len(q)
    W = sum(q)
    U = (x0 * W) >> 32
    C = np.cumsum(np.array(q, dtype=object))
    out = []
    for k in range(N):
        point = Fraction(k * W + U, N)
        out.append(next(i for i in range(N) if Fraction(int(C[i])) > point))
    return out


def test_brute_force_small_N_all_offset_buckets(oracle):
    rng = np.random.default_rng(5)
    for N in (1, 2, 3, 4):
        for trial in range(6):
            v = rng.uniform(0, 1, N).astype(np.float32)
            v[rng.integers(0, N)] = 1.0
            if trial == 0 and N > 1:
                v[0] = 0.0
            # sweep offsets finely enough to visit every bucket of the comb, plus both ends
            x0s = list(range(0, 2 ** 32, 2 ** 32 // 257)) + [2 ** 32 - 1]
            for x0 in x0s:
                anc, st = oracle.resample_systematic_x0(v, x0)
                assert st == 0
                assert list(anc) == _brute(v, x0)


def test_count_form_equivalence(oracle):
    """cnt_i = F(N C_i) - F(N C_{i-1}), F(X) = clamp(ceil((X - U)/W), 0, N)."""
    rng = np.random.default_rng(8)
    N = 513
    v = np.exp(2 * rng.standard_normal(N)).astype(np.float32)
    v /= v.max()
    q = _quant(v)
    W = sum(q)
    for x0 in X0S:
        U = (x0 * W) >> 32
        anc, _ = oracle.resample_systematic_x0(v, x0)
        cnt = _counts(anc, N)

        def F(X):
            return min(max(-((U - X) // W), 0), N)      # ceil((X-U)/W)
        C = 0
        for i in range(N):
            prev = C
            C += q[i]
            assert cnt[i] == F(N * C) - F(N * prev)


def test_seeded_entry_uses_stream4_word(oracle):
    rng = np.random.default_rng(2)
    v = rng.uniform(0, 1, 300).astype(np.float32)
    v[7] = 1.0
    for seed in (0, 1, 0xDEADBEEFCAFE):
        a, _ = oracle.resample_systematic(v, seed)
        b, _ = oracle.resample_systematic_x0(v, oracle.resample_word(seed))
        assert np.array_equal(a, b)


def test_normalised_weights_sum_to_one(oracle):
    rng = np.random.default_rng(4)
    for N in (1, 10, 100000):
        v = np.exp(2 * rng.standard_normal(N)).astype(np.float32)
        v /= v.max()
        w, st = oracle.normalised_weights(v)
        assert st == 0
        assert abs(w.sum() - 1.0) < 1e-12 * max(1, N)
        # the quantisation moves a weight by at most 2^-32 of the maximum
        assert np.max(np.abs(w - v.astype(np.float64) / v.astype(np.float64).sum())) < 2.0 ** -31
    w, st = oracle.normalised_weights(np.zeros(4, np.float32))
    assert st == -2


@pytest.mark.parametrize("N", [1 << 20])
def test_large_N_invariants(oracle, N):
    """Config 4 scale (2^20 particles, log-weights ~ N(0, 4))."""
    rng = np.random.default_rng(9)
    g = 2.0 * rng.standard_normal(N)
    v = np.exp(g - g.max()).astype(np.float32)
    anc, st = oracle.resample_systematic_x0(v, 0x9E3779B9)
    assert st == 0
    cnt = _counts(anc, N)
    assert cnt.sum() == N and np.all(np.diff(anc) >= 0)
    q = np.floor(v.astype(np.float64) * 2.0 ** 32)
    expect = N * q / q.sum()
    assert np.all(np.abs(cnt - expect) < 1.0 + 1e-6)
