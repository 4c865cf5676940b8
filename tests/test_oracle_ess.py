"""Pins for the oracle's adaptive (ESS-triggered) resampling.  CPU only.

The effective sample size has closed forms (uniform -> N, one-hot -> 1, k equal weights -> k, scale
invariance, the textbook identity ESS = 1 / sum wbar_i^2 for normalised weights); the adaptive update
must agree with the separately pinned plain update on everything the decision does not touch, equal
it bit for bit when it resamples, and carry the normalised weights forward when it does not."""
import numpy as np

from paper_2606_19729_b200 import synth


def test_ess_closed_forms(oracle):
    N = 1000
    assert oracle.effective_sample_size(np.full(N, 0.3, np.float32)) == np.float64(N) or \
        abs(oracle.effective_sample_size(np.full(N, 0.3, np.float32)) - N) < 1e-6 * N
    v = np.zeros(N, np.float32)
    v[17] = 0.8
    assert abs(oracle.effective_sample_size(v) - 1.0) < 1e-12
    for k in (2, 7, 250):
        v = np.zeros(N, np.float32)
        v[:k] = 0.125                      # exactly representable: k equal weights
        assert abs(oracle.effective_sample_size(v) - k) < 1e-9 * k
    assert oracle.effective_sample_size(np.zeros(5, np.float32)) == 0.0
    # a hand case: weights (1, 2, 3) / 8 -> (6/8)^2 / (14/64) = 36/14
    v = np.array([1, 2, 3], np.float32) / 8
    assert abs(oracle.effective_sample_size(v) - 36.0 / 14.0) < 1e-12


def test_ess_scale_invariance_and_textbook_identity(oracle):
    rng = np.random.default_rng(5)
    v = np.exp(rng.standard_normal(4096)).astype(np.float32)
    v /= v.max()
    e1 = oracle.effective_sample_size(v)
    e2 = oracle.effective_sample_size((v * np.float32(0.25)).astype(np.float32))  # exact scaling
    assert abs(e1 - e2) < 1e-9 * e1
    wbar = v.astype(np.float64) / v.astype(np.float64).sum()
    assert abs(e1 - 1.0 / np.sum(wbar ** 2)) < 1e-9 * e1
    assert 1.0 <= e1 <= v.size


def _case(lam):
    cfg = synth.CONFIGS[2]
    model = synth.make_model(cfg, prec=synth.PREC_FP32, lam=lam)
    inp = synth.make_inputs(cfg, N=600, P=8, Q=1, H=1)
    return model, inp


def test_adaptive_update_matches_plain_update(oracle):
    model, inp = _case(1.0)
    om = oracle.OracleModel(model)
    plain = om.belief_update(inp.bu_particles, 1, inp.observation, None, 99)
    ess = oracle.effective_sample_size(plain["post_weights"])
    # threshold above ESS/N: resamples -> identical to the plain update, bit for bit
    hi = om.belief_update(inp.bu_particles, 1, inp.observation, None, 99, ess_threshold=min(1.0, ess / 600 * 1.5 + 0.01))
    assert hi["resampled"] == 1 and abs(hi["ess"] - ess) < 1e-9 * ess
    for k in ("ancestors", "particles", "weights", "post_weights", "proposals"):
        assert np.array_equal(hi[k], plain[k]), k
    # threshold below ESS/N: keeps the proposals, carries the normalised weights
    lo = om.belief_update(inp.bu_particles, 1, inp.observation, None, 99, ess_threshold=ess / 600 * 0.5)
    assert lo["resampled"] == 0 and lo["status"] == 0
    assert np.array_equal(lo["ancestors"], np.arange(600))
    assert np.array_equal(lo["particles"], plain["proposals"])
    v = plain["post_weights"].astype(np.float64)
    assert np.allclose(lo["weights"], v / v.sum(), rtol=1e-6, atol=0)
    assert abs(float(lo["weights"].astype(np.float64).sum()) - 1.0) < 1e-5
    assert lo["log_evidence"] == plain["log_evidence"]


def test_flat_likelihood_keeps_ess_at_n(oracle):
    """lambda -> infinity flattens the likelihood: weights uniform, ESS = N, no
    resampling for any threshold below 1."""
    model, inp = _case(1e30)
    om = oracle.OracleModel(model)
    o = om.belief_update(inp.bu_particles, 1, inp.observation, None, 3, ess_threshold=0.999)
    assert o["resampled"] == 0 and abs(o["ess"] - 600.0) < 1e-6
    assert np.allclose(o["weights"], 1.0 / 600.0, rtol=1e-6)


def test_degenerate_weights_never_resample(oracle):
    model, inp = _case(1.0)
    om = oracle.OracleModel(model)
    o = om.belief_update(inp.bu_particles, 0, inp.observation, np.zeros(600, np.float32), 1, ess_threshold=0.5)
    assert o["status"] != 0 and o["resampled"] == 0 and o["ess"] == 0.0
    assert np.array_equal(o["ancestors"], np.arange(600))
