"""Pins for the oracle's SIR belief update (O5).  CPU only.

Expected values: the exponential-tilt closed form of a Gaussian proposal under a log-linear
likelihood (SURVEY 8c pin 5), scipy.special.logsumexp (library), invariances the paper states
(only relative weights matter), and a step-by-step recomposition from the separately
pinned pieces (MLP forward, noise, resampler).
"""
import pytest
import numpy as np
import scipy.special

from paper_2606_19729_b200 import synth
from paper_2606_19729_b200.synth import ACT_NONE, MLPSpec, ModelSpec, R_NEG_L2_GOAL


def _linear_bu_model(rng, S, O, A, Nz, lam):
    gin = S + A + Nz
    WT = (rng.standard_normal((S, gin)) * 0.5).astype(np.float32)
    bT = (rng.standard_normal(S) * 0.1).astype(np.float32)
    f_T = MLPSpec([gin, S], ACT_NONE, [WT], [bT])
    f_Z = synth.make_mlp(rng, [gin, O], ACT_NONE)
    d = 5
    lik_obs = MLPSpec([O, d], ACT_NONE, [(rng.standard_normal((d, O)) * 0.4).astype(np.float32)],
                      [(rng.standard_normal(d) * 0.1).astype(np.float32)])
    lik_state = MLPSpec([S, d], ACT_NONE, [(rng.standard_normal((d, S)) * 0.4).astype(np.float32)],
                        [(rng.standard_normal(d) * 0.1).astype(np.float32)])
    return ModelSpec(S, O, A, Nz, f_T, f_Z, lik_obs, lik_state, lam=lam, gamma=0.9,
                     reward_kind=R_NEG_L2_GOAL, reward_param=np.zeros(S, np.float32))


def test_exponential_tilt_closed_form(oracle):
    """Particles ~ N(0, I), linear f_T and linear towers: proposals are N(mu, Sig) with
    mu = B e_a + b, Sig = A A^T + C C^T, log-likelihood l = c + h0^T s', so the posterior is
    N(mu + Sig h, Sig) with h = h0/lambda and log evidence = c/lambda + h^T mu + h^T Sig h / 2."""
    rng = np.random.default_rng(10)
    S, O, A, Nz, lam, N, a = 3, 4, 3, 2, 1.25, 1 << 16, 2
    m = _linear_bu_model(rng, S, O, A, Nz, lam)
    om = oracle.OracleModel(m)
    particles = rng.standard_normal((N, S)).astype(np.float32)
    obs = rng.standard_normal(O).astype(np.float32)
    out = om.belief_update(particles, a, obs, None, seed=2024)
    assert out["status"] == 0
    WT = m.f_T.W[0].astype(np.float64)
    Am, Bm, Cm, bT = WT[:, :S], WT[:, S:S + A], WT[:, S + A:], m.f_T.b[0].astype(np.float64)
    mu = Bm[:, a] + bT
    Sig = Am @ Am.T + Cm @ Cm.T
    e = m.lik_obs.W[0].astype(np.float64) @ obs + m.lik_obs.b[0]
    G, g0 = m.lik_state.W[0].astype(np.float64), m.lik_state.b[0].astype(np.float64)
    h = G.T @ e / lam
    c = e @ g0 / lam
    post_mu = mu + Sig @ h
    logev = c + h @ mu + 0.5 * h @ Sig @ h
    # proposals really are N(mu, Sig)
    prop = out["proposals"].astype(np.float64)
    assert np.all(np.abs(prop.mean(0) - mu) < 5 * np.sqrt(np.diag(Sig) / N))
    np.testing.assert_allclose(np.cov(prop.T), Sig, atol=0.03 * np.abs(Sig).max())
    # posterior moments after resampling; tilt strength makes the ESS < N, so allow 1.5 %
    post = out["particles"].astype(np.float64)
    scale = np.sqrt(np.diag(Sig))
    assert np.all(np.abs(post.mean(0) - post_mu) < 0.015 * scale * max(1.0, np.linalg.norm(h)) + 0.01)
    np.testing.assert_allclose(np.cov(post.T), Sig, atol=0.05 * np.abs(Sig).max())
    assert abs(out["log_evidence"] - logev) < 0.02
    # the shift moved the mean by something measurable (the test has power)
    assert np.linalg.norm(post_mu - mu) > 0.1
    assert np.allclose(out["weights"], 1.0 / N)


def test_recomposition_from_pinned_pieces(oracle):
    for lik_action_cond in (0, 1):
        cfg = synth.CONFIGS[1]
        m = synth.make_model(cfg, lik_action_cond=lik_action_cond, lam=1.25)
        om = oracle.OracleModel(m)
        inp = synth.make_inputs(cfg)
        N, a, seed = cfg.N, 3, 555
        rng = np.random.default_rng(0)
        w = rng.uniform(0.0, 2.0, N).astype(np.float32)
        w[5] = 0.0
        out = om.belief_update(inp.bu_particles, a, inp.observation, w, seed)
        # proposals = f_T([s ; onehot(a) ; omega(i,0,0; stream 3)])
        x = np.zeros((N, cfg.S + cfg.A + cfg.Nz), np.float32)
        x[:, :cfg.S] = inp.bu_particles
        x[:, cfg.S + a] = 1.0
        for i in range(N):
            x[i, cfg.S + cfg.A:] = oracle.normals(seed, i, 0, 0, 3, cfg.Nz)
        prop = om.mlp_forward(0, x)
        assert np.array_equal(prop, out["proposals"])
        e = om.mlp_forward(2, inp.observation[None, :])[0]
        gin = prop
        if lik_action_cond:
            oh = np.zeros((N, cfg.A), np.float32)
            oh[:, a] = 1.0
            gin = np.concatenate([prop, oh], axis=1)
        ell = om.mlp_forward(3, gin).astype(np.float64) @ e.astype(np.float64)
        with np.errstate(divide="ignore"):
            L = np.log(w.astype(np.float64)) + ell / 1.25
        np.testing.assert_allclose(out["logits"][w > 0], L[w > 0], rtol=2e-5, atol=2e-5)
        assert out["logits"][5] == -np.inf and out["post_weights"][5] == 0.0
        v = np.exp(out["logits"].astype(np.float64) - out["logits"].max())
        np.testing.assert_allclose(out["post_weights"], v, rtol=3e-6, atol=1e-30)
        assert out["post_weights"].max() == 1.0
        anc, st = oracle.resample_systematic(out["post_weights"], seed)
        assert st == 0 and np.array_equal(anc, out["ancestors"])
        assert np.array_equal(out["particles"], prop[anc])
        # log evidence = logsumexp(L) - log(sum w)   (library: scipy)
        ref = scipy.special.logsumexp(out["logits"].astype(np.float64)) - np.log(w.astype(np.float64).sum())
        assert abs(out["log_evidence"] - ref) < 1e-6 * max(1.0, abs(ref))


def test_only_relative_weights_matter(oracle):
    """scaling every prior weight (= adding a constant to every L_i) leaves the
    normalised weights and the resampling unchanged up to rounding of the shift."""
    cfg = synth.CONFIGS[2]
    m = synth.make_model(cfg)
    om = oracle.OracleModel(m)
    inp = synth.make_inputs(cfg, N=2048)
    rng = np.random.default_rng(1)
    w = np.exp(rng.standard_normal(2048)).astype(np.float32)
    a = om.belief_update(inp.bu_particles, 1, inp.observation, w, 3)
    b = om.belief_update(inp.bu_particles, 1, inp.observation, 8.0 * w, 3)   # exact power of two
    np.testing.assert_allclose(a["post_weights"], b["post_weights"], rtol=1e-5, atol=1e-12)
    assert np.mean(a["ancestors"] != b["ancestors"]) < 0.01
    assert abs(a["log_evidence"] - b["log_evidence"]) < 1e-5


def test_lambda_to_infinity_gives_prior(oracle):
    cfg = synth.CONFIGS[1]
    m = synth.make_model(cfg, lam=1e12)
    om = oracle.OracleModel(m)
    inp = synth.make_inputs(cfg)
    out = om.belief_update(inp.bu_particles, 0, inp.observation, None, 17)
    assert np.allclose(out["post_weights"], 1.0, atol=1e-6)
    assert np.array_equal(out["ancestors"], np.arange(cfg.N))
    assert abs(out["log_evidence"]) < 1e-6


def test_large_scores_do_not_overflow(oracle):
    """max-shifted log-sum-exp: scores up to +-1e4 stay finite."""
    cfg = synth.CONFIGS[1]
    m = synth.make_model(cfg, lam=1e-3)          # l / lambda of order 1e3..1e4
    om = oracle.OracleModel(m)
    inp = synth.make_inputs(cfg)
    out = om.belief_update(inp.bu_particles, 0, inp.observation, None, 17)
    assert out["status"] == 0 and np.isfinite(out["log_evidence"])
    assert np.abs(out["logits"]).max() > 100
    assert out["post_weights"].max() == 1.0 and np.all(np.isfinite(out["post_weights"]))
    ref = scipy.special.logsumexp(out["logits"].astype(np.float64)) - np.log(cfg.N)
    assert abs(out["log_evidence"] - ref) < 1e-6 * abs(ref)


def test_all_zero_prior_weights_pass_through(oracle):
    cfg = synth.CONFIGS[1]
    m = synth.make_model(cfg)
    om = oracle.OracleModel(m)
    inp = synth.make_inputs(cfg)
    out = om.belief_update(inp.bu_particles, 0, inp.observation, np.zeros(cfg.N, np.float32), 1)
    assert out["status"] == -2
    assert np.array_equal(out["ancestors"], np.arange(cfg.N))
    assert np.array_equal(out["particles"], out["proposals"])


@pytest.mark.parametrize("bad", ["nan_state", "inf_weight"])
def test_nonfinite_score_is_flagged(oracle, bad):
    """Reading R20: any non-finite L_i (a NaN that a particle's state carried through
    f_T and g, or +inf from an infinite prior weight) makes the update degenerate: non-zero status,
    identity ancestors, particles_out = proposals, weights 1/N, log-evidence -inf; it never leaks
    into the resampler.  (A NaN prior WEIGHT is not > 0 and counts as a zero weight.)"""
    cfg = synth.CONFIGS[2]
    om = oracle.OracleModel(synth.make_model(cfg))
    N = 300
    inp = synth.make_inputs(cfg, N=N)
    w = np.full(N, 1.0 / N, np.float32)
    parts = inp.bu_particles.copy()
    if bad == "nan_state":
        parts[17, 3] = np.nan
    else:
        w[17] = np.inf
    out = om.belief_update(parts, 2, inp.observation, w, 11)
    assert out["status"] != 0
    assert (np.isnan(out["logits"][17]) if bad == "nan_state" else np.isposinf(out["logits"][17]))
    assert np.array_equal(out["ancestors"], np.arange(N))
    assert np.array_equal(out["particles"], out["proposals"], equal_nan=True)
    assert np.all(out["weights"] == np.float32(1.0) / np.float32(N))
    assert np.isneginf(out["log_evidence"])
    # a NaN prior weight is a zero weight: the update stays regular and never picks that particle
    w[17] = np.nan
    out = om.belief_update(inp.bu_particles, 2, inp.observation, w, 11)
    assert out["status"] == 0 and not np.any(out["ancestors"] == 17)
