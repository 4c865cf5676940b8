"""Pins for the oracle's rollout value estimate (O4).  CPU only.

Expected values come from closed forms, from brute-force enumeration written independently here
(numpy fp64 on top of the KAT-pinned noise words), and from invariants: see SURVEY.md 8(c)
"Pins with no implementation to compare against" 1-4, 9.
"""
import numpy as np

from paper_2606_19729_b200 import synth
from paper_2606_19729_b200.synth import (ACT_NONE, ACT_RELU, ACT_SILU, MLPSpec, ModelSpec,
                                         R_LINEAR, R_NEG_L2_GOAL, R_NEG_QUADRATIC)


def _towers(rng, S, O):
    return (synth.make_mlp(rng, [O, 4, 3], ACT_NONE), synth.make_mlp(rng, [S, 4, 3], ACT_NONE))


def _linear_model(rng, S, O, A, Nz, gamma, noise_scale, reward_kind, reward_param, cost=None):
    """f_T(s,a,w) = A s + B e_a + C w + b (single affine layer), f_Z likewise."""
    gin = S + A + Nz
    WT = (rng.standard_normal((S, gin)) * 0.4).astype(np.float32)
    WT[:, S + A:] *= noise_scale
    bT = (rng.standard_normal(S) * 0.1).astype(np.float32)
    WZ = (rng.standard_normal((O, gin)) * 0.4).astype(np.float32)
    WZ[:, S + A:] *= noise_scale
    bZ = (rng.standard_normal(O) * 0.1).astype(np.float32)
    f_T = MLPSpec([gin, S], ACT_NONE, [WT], [bT])
    f_Z = MLPSpec([gin, O], ACT_NONE, [WZ], [bZ])
    lo, ls = _towers(rng, S, O)
    return ModelSpec(S, O, A, Nz, f_T, f_Z, lo, ls, gamma=gamma, reward_kind=reward_kind,
                     reward_param=reward_param, action_cost=cost)


def test_deterministic_linear_generator_closed_form(oracle):
    """C = 0: s_t = A^t s_0 + sum_k A^(t-1-k) (B e_{a_k} + b); linear reward c^T s + c0 + cost[a]."""
    rng = np.random.default_rng(1)
    S, O, A, Nz, H, P, Q, gamma = 3, 2, 4, 2, 7, 5, 6, 0.9
    c = rng.standard_normal(S + 1).astype(np.float32)
    cost = rng.uniform(-0.3, 0, A).astype(np.float32)
    m = _linear_model(rng, S, O, A, Nz, gamma, 0.0, R_LINEAR, c, cost)
    om = oracle.OracleModel(m)
    particles = rng.standard_normal((P, S)).astype(np.float32)
    seqs = rng.integers(0, A, (Q, H), dtype=np.int32)
    w = rng.uniform(0.1, 2.0, P).astype(np.float32)
    V, Wit, G = om.rollout_values(particles, seqs, w, seed=77, want_returns=True)
    WT = m.f_T.W[0].astype(np.float64)
    Am, Bm, bT = WT[:, :S], WT[:, S:S + A], m.f_T.b[0].astype(np.float64)
    WZ = m.f_Z.W[0].astype(np.float64)
    Az, Bz, bZ = WZ[:, :S], WZ[:, S:S + A], m.f_Z.b[0].astype(np.float64)
    wbar = w.astype(np.float64) / w.astype(np.float64).sum()
    Vref = np.zeros(Q)
    Witref = np.zeros((Q, O))
    Gref = np.zeros((Q, P))
    for q in range(Q):
        for p in range(P):
            s = particles[p].astype(np.float64)
            for t in range(H):
                a = seqs[q, t]
                Gref[q, p] += gamma ** t * (c[:S].astype(np.float64) @ s + c[S] + cost[a])
                s = Am @ s + Bm[:, a] + bT
                Witref[q] += wbar[p] * gamma ** t * (Az @ s + Bz[:, a] + bZ)
        Vref[q] = wbar @ Gref[q]
    np.testing.assert_allclose(G, Gref, rtol=2e-5, atol=2e-5)
    np.testing.assert_allclose(V, Vref, rtol=2e-5, atol=2e-5)
    np.testing.assert_allclose(Wit, Witref, rtol=2e-5, atol=2e-5)
    # closed form with matrix powers for the final state of one (p,q)
    _, states, _ = om.rollout_trajectory(particles[2], seqs[3], 2, 3, 77)
    sH = np.linalg.matrix_power(Am, H) @ particles[2].astype(np.float64)
    for k in range(H):
        sH += np.linalg.matrix_power(Am, H - 1 - k) @ (Bm[:, seqs[3, k]] + bT)
    np.testing.assert_allclose(states[H], sH, rtol=2e-5, atol=2e-5)


def test_identity_relu_generator_keeps_particles(oracle):
    """s = relu(s) - relu(-s) with hidden width 2S: the rollout leaves particles unchanged, so
    V_q = sum_p wbar_p R(s_p) (1 - gamma^H)/(1 - gamma) for a state-only reward."""
    rng = np.random.default_rng(2)
    S, O, A, Nz, H, P, Q, gamma = 4, 3, 3, 2, 9, 33, 4, 0.95
    gin = S + A + Nz
    W1 = np.zeros((2 * S, gin), np.float32)
    W1[:S, :S] = np.eye(S)
    W1[S:, :S] = -np.eye(S)
    W2 = np.concatenate([np.eye(S), -np.eye(S)], axis=1).astype(np.float32)
    f_T = MLPSpec([gin, 2 * S, S], ACT_RELU, [W1, W2], [np.zeros(2 * S, np.float32), np.zeros(S, np.float32)])
    f_Z = synth.make_mlp(rng, [gin, 8, O], ACT_RELU)
    lo, ls = _towers(rng, S, O)
    goal = rng.uniform(-1, 1, S).astype(np.float32)
    m = ModelSpec(S, O, A, Nz, f_T, f_Z, lo, ls, gamma=gamma, reward_kind=R_NEG_L2_GOAL,
                  reward_param=goal)
    om = oracle.OracleModel(m)
    particles = rng.standard_normal((P, S)).astype(np.float32)
    seqs = rng.integers(0, A, (Q, H), dtype=np.int32)
    w = rng.uniform(0.1, 1, P).astype(np.float32)
    V, _ = om.rollout_values(particles, seqs, w, seed=5)
    R = -np.linalg.norm(particles.astype(np.float64) - goal, axis=1)
    wbar = w.astype(np.float64) / w.astype(np.float64).sum()
    expect = (wbar @ R) * (1 - gamma ** H) / (1 - gamma)
    np.testing.assert_allclose(V, np.full(Q, expect), rtol=1e-5)
    _, states, _ = om.rollout_trajectory(particles[0], seqs[0], 0, 0, 5)
    assert np.array_equal(states[-1], particles[0])


def test_constant_reward_pins_discount_indexing(oracle):
    """R = c0: V_q = c0 (1 - gamma^H)/(1 - gamma) for every q (gamma^t with t from 0, H terms)."""
    rng = np.random.default_rng(3)
    cfg = synth.CONFIGS[1]
    for gamma, H in [(0.95, 10), (0.5, 3), (1.0, 4)]:
        c = np.zeros(cfg.S + 1, np.float32)
        c[-1] = -2.5
        m = synth.make_model(cfg).replace(gamma=gamma, reward_kind=R_LINEAR, reward_param=c)
        om = oracle.OracleModel(m)
        particles = rng.standard_normal((16, cfg.S)).astype(np.float32)
        seqs = rng.integers(0, cfg.A, (5, H), dtype=np.int32)
        V, _ = om.rollout_values(particles, seqs, None, seed=1)
        geo = H if gamma == 1.0 else (1 - gamma ** H) / (1 - gamma)
        np.testing.assert_allclose(V, np.full(5, -2.5 * geo), rtol=1e-6)


def _np_mlp(f, x):
    h = np.asarray(x, np.float64)
    for l in range(f.n_layers):
        h = f.W[l].astype(np.float64) @ h + f.b[l].astype(np.float64)
        if l < f.n_layers - 1:
            if f.act == ACT_RELU:
                h = np.maximum(h, 0)
            elif f.act == ACT_SILU:
                h = h / (1 + np.exp(-h))
    return h


def _onehot(a, A):
    e = np.zeros(A)
    e[a] = 1
    return e


def test_depth2_brute_force_enumeration(oracle):
    """A = 4, H = 2, all 16 sequences: V(a0 a1) = sum_p wbar_p [R(s_p,a0) + gamma R(f_T(s_p,a0,w),a1)]
    written as an independent recursion in numpy fp64 using the same (KAT-pinned) noise."""
    rng = np.random.default_rng(4)
    cfg = synth.CONFIGS[1]
    m = synth.make_model(cfg, action_cost=True)
    om = oracle.OracleModel(m)
    P, A, S, seed = 7, cfg.A, cfg.S, 424242
    particles = rng.standard_normal((P, S)).astype(np.float32)
    w = rng.uniform(0.2, 1.0, P).astype(np.float32)
    seqs = np.array([[a0, a1] for a0 in range(A) for a1 in range(A)], dtype=np.int32)
    V, Wit = om.rollout_values(particles, seqs, w, seed=seed)
    goal = m.reward_param.astype(np.float64)
    cost = m.action_cost.astype(np.float64)

    def R(s, a):
        return -np.linalg.norm(s - goal) + cost[a]
    wbar = w.astype(np.float64) / w.astype(np.float64).sum()
    for q, (a0, a1) in enumerate(seqs):
        v = 0.0
        wit = np.zeros(cfg.O)
        for p in range(P):
            s0 = particles[p].astype(np.float64)
            om_T0 = oracle.normals(seed, p, q, 0, 1, cfg.Nz)
            s1 = _np_mlp(m.f_T, np.concatenate([s0, _onehot(a0, A), om_T0]))
            om_Z0 = oracle.normals(seed, p, q, 0, 2, cfg.Nz)
            o1 = _np_mlp(m.f_Z, np.concatenate([s1, _onehot(a0, A), om_Z0]))
            om_T1 = oracle.normals(seed, p, q, 1, 1, cfg.Nz)
            s2 = _np_mlp(m.f_T, np.concatenate([s1, _onehot(a1, A), om_T1]))
            om_Z1 = oracle.normals(seed, p, q, 1, 2, cfg.Nz)
            o2 = _np_mlp(m.f_Z, np.concatenate([s2, _onehot(a1, A), om_Z1]))
            v += wbar[p] * (R(s0, a0) + m.gamma * R(s1, a1))
            wit += wbar[p] * (o1 + m.gamma * o2)
        assert abs(V[q] - v) < 2e-5 * max(1.0, abs(v))
        np.testing.assert_allclose(Wit[q], wit, rtol=2e-5, atol=2e-5)
    # PORPP-style soft value over the root actions computed both ways
    eta = 2.0
    Vm = V.reshape(A, A).astype(np.float64)
    psi = Vm.max(axis=1)
    soft = np.log(np.exp(eta * (psi - psi.max())).sum()) / eta + psi.max()
    import scipy.special
    assert abs(soft - scipy.special.logsumexp(eta * psi) / eta) < 1e-12


def test_q_offset_slices_reproduce_full_run(oracle):
    cfg = synth.CONFIGS[1]
    m = synth.make_model(cfg)
    om = oracle.OracleModel(m)
    inp = synth.make_inputs(cfg, P=24, Q=10, H=4)
    V, Wit = om.rollout_values(inp.particles, inp.action_seqs, None, seed=9)
    V2, Wit2 = om.rollout_values(inp.particles, inp.action_seqs[6:], None, seed=9, q_offset=6)
    assert np.array_equal(V[6:], V2) and np.array_equal(Wit[6:], Wit2)


def test_stochastic_linear_moments(oracle):
    """s' = A s + B e_a + C w + b with w ~ N(0, I): mean and covariance of s_t in closed form,
    E[-s^T M s] = -(mu^T M mu + tr(M Sigma)); the MC estimate over P particles is within 5 sigma."""
    rng = np.random.default_rng(6)
    S, O, A, Nz, H, P, gamma = 3, 2, 2, 3, 4, 20000, 0.9
    B = rng.standard_normal((S, S))
    M = (B @ B.T / S).astype(np.float32)
    m = _linear_model(rng, S, O, A, Nz, gamma, 1.0, R_NEG_QUADRATIC, M)
    om = oracle.OracleModel(m)
    s0 = rng.standard_normal(S).astype(np.float32)
    particles = np.tile(s0, (P, 1))
    seqs = np.array([[0, 1, 1, 0]], dtype=np.int32)
    V, _, G = om.rollout_values(particles, seqs, None, seed=31337, want_returns=True)
    WT = m.f_T.W[0].astype(np.float64)
    Am, Bm, Cm, bT = WT[:, :S], WT[:, S:S + A], WT[:, S + A:], m.f_T.b[0].astype(np.float64)
    mu, Sig = s0.astype(np.float64), np.zeros((S, S))
    Md = M.astype(np.float64)
    expect = 0.0
    for t in range(H):
        expect += gamma ** t * -(mu @ Md @ mu + np.trace(Md @ Sig))
        mu = Am @ mu + Bm[:, seqs[0, t]] + bT
        Sig = Am @ Sig @ Am.T + Cm @ Cm.T
    se = G[0].astype(np.float64).std() / np.sqrt(P)
    assert abs(V[0] - expect) < 5 * se
    assert se < 0.05 * abs(expect)       # the test has power: a dropped term would show
    # final-state moments from the per-particle trajectories of a subsample
    fin = np.array([om.rollout_trajectory(s0, seqs[0], p, 0, 31337)[1][-1] for p in range(4000)])
    assert np.all(np.abs(fin.mean(0) - mu) < 5 * np.sqrt(np.diag(Sig) / 4000))
    np.testing.assert_allclose(np.cov(fin.T), Sig, atol=6 * np.abs(Sig).max() / np.sqrt(4000))


def test_noise_off_duplicate_sequences_bit_identical(oracle):
    cfg = synth.CONFIGS[2]
    m = synth.make_model(cfg)
    for f in (m.f_T, m.f_Z):
        f.W[0][:, cfg.S + cfg.A:] = 0.0
    om = oracle.OracleModel(m)
    inp = synth.make_inputs(cfg, P=16, Q=4, H=5)
    seqs = inp.action_seqs.copy()
    seqs[3] = seqs[1]
    V, Wit = om.rollout_values(inp.particles, seqs, None, seed=3)
    assert V[3] == V[1] and np.array_equal(Wit[3], Wit[1])
    V2, _ = om.rollout_values(inp.particles, seqs, None, seed=999)      # seed irrelevant now
    assert np.array_equal(V, V2)


def test_values_are_weighted_means_of_returns(oracle):
    cfg = synth.CONFIGS[2]
    m = synth.make_model(cfg)
    om = oracle.OracleModel(m)
    inp = synth.make_inputs(cfg, P=50, Q=3, H=6)
    rng = np.random.default_rng(1)
    w = rng.uniform(0, 3, 50).astype(np.float32)
    w[4] = 0.0
    V, _, G = om.rollout_values(inp.particles, inp.action_seqs, w, seed=8, want_returns=True)
    wb = w.astype(np.float64) / w.astype(np.float64).sum()
    np.testing.assert_allclose(V, G.astype(np.float64) @ wb, rtol=1e-6)
    # unnormalised weights: scaling leaves values unchanged; None == uniform
    V3, _ = om.rollout_values(inp.particles, inp.action_seqs, 4 * w, seed=8)
    np.testing.assert_allclose(V3, V, rtol=1e-6)
    Vu, _ = om.rollout_values(inp.particles, inp.action_seqs, None, seed=8)
    Vo, _ = om.rollout_values(inp.particles, inp.action_seqs, np.ones(50, np.float32), seed=8)
    assert np.array_equal(Vu, Vo)


def test_f32_oracle_close_to_f64_build(oracle):
    """How far fp32 arithmetic itself is from exact: bounds the tolerance the GPU fp32 mode is held
    to (north_star: relative 1e-4)."""
    for idx in (1, 2):
        cfg = synth.CONFIGS[idx]
        m = synth.make_model(cfg)
        inp = synth.make_inputs(cfg, P=32, Q=4, H=cfg.H)
        V32, W32 = oracle.OracleModel(m, "f32").rollout_values(inp.particles, inp.action_seqs, None, 7)
        V64, W64 = oracle.OracleModel(m, "f64").rollout_values(inp.particles, inp.action_seqs, None, 7)
        assert np.max(np.abs(V32 - V64)) < 2e-6 * np.max(np.abs(V64))
        assert np.max(np.abs(W32 - W64)) < 2e-5 * np.max(np.abs(W64))
