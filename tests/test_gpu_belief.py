"""GPU parity: voila_belief_update / voila_resample_systematic / voila_mlp_forward (through the
C ABI) against the CPU oracle.  Indices must be bit-exact given identical weights (north_star):
the GPU's own post_weights array is fed to the oracle's exact-integer resampler (SURVEY 8c O7
test protocol).  Run on the B200 box: pytest -m gpu."""
import numpy as np
import pytest

from paper_2606_19729_b200 import synth
from tests.parity_util import TOL_BF16_STATE, TOL_FP32, assert_close, rel_inf, t2n

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _gpu_bu(torch, model, particles, action, obs, weights, seed, prec, kernel=0):
    import paper_2606_19729_b200 as vl
    ctx = vl.Voila(model, device=0, prec=prec)
    if kernel in (vl.KERNEL_TCGEN05, vl.KERNEL_TCGEN05_PAIR) and not ctx.voila_tcgen05_supported():
        ctx.close()
        pytest.skip("tcgen05 path does not support these dims")
    ctx.voila_set_kernel(kernel)
    parts = ctx.to_particles(particles)
    o = torch.from_numpy(obs).cuda()
    w = None if weights is None else torch.from_numpy(weights).cuda()
    out = ctx.voila_belief_update(parts, action, o, w, seed)
    torch.cuda.synchronize()
    if kernel == vl.KERNEL_TCGEN05_PAIR:  # the tensor-core program really ran (no silent CUDA-core fallback)
        assert ctx.voila_last_belief_kernel().startswith("belief_tc2_")
    res = {k: t2n(v) if v.dtype != torch.int32 else v.cpu().numpy() for k, v in out.items()}
    ctx.close()
    return res


def _check_bu(oracle, model, particles, action, obs, weights, seed, g, tol, bf16):
    om = oracle.OracleModel(model)
    parts = synth.bf16_round_np(particles) if bf16 else particles
    o = om.belief_update(parts, action, obs, weights, seed)
    N = particles.shape[0]
    assert int(g["status"][0]) == 0 and o["status"] == 0
    assert_close(g["proposals"], o["proposals"], tol, "proposals")
    # v_i = exp(L_i - m) in [0,1]: absolute error (relative to the max, which is 1)
    assert rel_inf(g["post_weights"], o["post_weights"]) <= (5e-2 if bf16 else 2e-4)
    assert abs(float(g["log_evidence"][0]) - o["log_evidence"]) <= (5e-2 if bf16 else 2e-4) * max(
        1.0, abs(o["log_evidence"]))
    # bit-exact indices given identical weights
    anc_ref, st = oracle.resample_systematic(g["post_weights"], seed)
    assert st == 0
    assert np.array_equal(g["ancestors"], anc_ref)
    assert np.all(np.diff(g["ancestors"]) >= 0)
    # the gather: particles_out[k] == proposals[ancestors[k]] exactly
    assert np.array_equal(g["particles"], g["proposals"][g["ancestors"]])
    assert np.all(g["weights"] == np.float32(1.0) / np.float32(N))
    mismatch = float(np.mean(g["ancestors"] != o["ancestors"]))
    return mismatch


@pytest.mark.parametrize("cfg_idx,N,use_w", [(1, 256, False), (1, 1, False), (2, 1000, True),
                                             (2, 2049, True), (3, 300, True)])
def test_belief_update_fp32(torch_cuda, oracle, cfg_idx, N, use_w):
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg, prec=synth.PREC_FP32, lam=1.25)
    inp = synth.make_inputs(cfg, N=N, P=8, Q=1, H=1)
    w = None
    if use_w:
        w = np.exp(2.0 * np.random.default_rng(3).standard_normal(N)).astype(np.float32)
        w[::5] = 0.0
    g = _gpu_bu(torch_cuda, model, inp.bu_particles, 1, inp.observation, w, 777, synth.PREC_FP32)
    mism = _check_bu(oracle, model, inp.bu_particles, 1, inp.observation, w, 777, g, TOL_FP32, False)
    assert mism <= 0.02  # reported, loosely bounded: end-to-end index agreement in fp32 mode
    if use_w:
        assert not np.any(np.isin(g["ancestors"], np.nonzero(w == 0)[0]))


def test_belief_update_action_conditioned_tower(torch_cuda, oracle):
    """lik_action_cond = 1: g's input is [s' ; onehot(a)] (reading R2)."""
    cfg = synth.CONFIGS[1]
    model = synth.make_model(cfg, prec=synth.PREC_FP32, lik_action_cond=1)
    inp = synth.make_inputs(cfg, N=500, P=8, Q=1, H=1)
    g = _gpu_bu(torch_cuda, model, inp.bu_particles, 3, inp.observation, None, 5, synth.PREC_FP32)
    _check_bu(oracle, model, inp.bu_particles, 3, inp.observation, None, 5, g, TOL_FP32, False)


@pytest.mark.parametrize("kernel_name", ["ffma", "tcgen05", "pair"])
@pytest.mark.parametrize("cfg_idx,N", [(2, 1024), (3, 2048), (4, 5000), (5, 700), (3, 1), (4, 255), (4, 257),
                                       (5, 40_001),
                                       # above 256 x 74 particles narrow models run the TWO-SLOT program
                                       (4, 40_001), (3, 19_000), (2, 65_536 + 300)])
def test_belief_update_bf16(torch_cuda, oracle, kernel_name, cfg_idx, N):
    import paper_2606_19729_b200 as vl
    kernel = {"ffma": vl.KERNEL_FFMA, "tcgen05": vl.KERNEL_TCGEN05, "pair": vl.KERNEL_TCGEN05_PAIR}[kernel_name]
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg, prec=synth.PREC_BF16)
    inp = synth.make_inputs(cfg, N=N, P=8, Q=1, H=1)
    g = _gpu_bu(torch_cuda, model, inp.bu_particles, 1, inp.observation, inp.bu_weights, 31,
                synth.PREC_BF16, kernel)
    _check_bu(oracle, model, inp.bu_particles, 1, inp.observation, inp.bu_weights, 31, g,
              TOL_BF16_STATE, True)


def test_belief_update_bf16_pair_variants(torch_cuda, oracle):
    """CTA-pair tcgen05 propose+score program: action-conditioned tower (one-hot folded into the
    bias of g's first layer), uniform prior (weights = NULL), another action and seed."""
    import paper_2606_19729_b200 as vl
    cfg = synth.CONFIGS[3]
    for cond, use_w, action, seed, N in [(1, False, 5, 99, 1500), (0, False, 0, 3, 1500), (1, True, 15, 1 << 40, 1500),
                                         (1, True, 7, 12345, 30_011)]:  # the last one: two-slot program
        model = synth.make_model(cfg, prec=synth.PREC_BF16, lik_action_cond=cond)
        inp = synth.make_inputs(cfg, N=N, P=8, Q=1, H=1)
        w = None
        if use_w:
            w = np.exp(2.0 * np.random.default_rng(4).standard_normal(N)).astype(np.float32)
            w[::7] = 0.0
        g = _gpu_bu(torch_cuda, model, inp.bu_particles, action, inp.observation, w, seed, synth.PREC_BF16,
                    vl.KERNEL_TCGEN05_PAIR)
        _check_bu(oracle, model, inp.bu_particles, action, inp.observation, w, seed, g, TOL_BF16_STATE, True)
        if use_w:
            assert not np.any(np.isin(g["ancestors"], np.nonzero(w == 0)[0]))


def test_belief_update_degenerate_weights(torch_cuda):
    """All prior weights zero: device status 1, ancestors = identity, particles_out = proposals."""
    cfg = synth.CONFIGS[1]
    model = synth.make_model(cfg)
    inp = synth.make_inputs(cfg, N=300, P=8, Q=1, H=1)
    w = np.zeros(300, np.float32)
    g = _gpu_bu(torch_cuda, model, inp.bu_particles, 0, inp.observation, w, 1, synth.PREC_FP32)
    assert int(g["status"][0]) == 1
    assert np.array_equal(g["ancestors"], np.arange(300))
    assert np.array_equal(g["particles"], g["proposals"])
    assert np.isneginf(g["log_evidence"][0])


@pytest.mark.parametrize("prec", [synth.PREC_FP32, synth.PREC_BF16])
@pytest.mark.parametrize("bad", ["nan_state", "inf_weight"])
def test_belief_update_nonfinite_score(torch_cuda, oracle, prec, bad):
    """Reading R20: a non-finite L_i (a NaN carried from one particle's state through f_T and g, or
    +inf from an infinite prior weight) gives device status 1 on the GPU and a non-zero status in the
    oracle, and the documented degenerate outputs: ancestors = identity, particles_out = proposals,
    weights 1/N, log-evidence -inf.  On the tensor-core path the NaN stays in its own accumulator row."""
    cfg = synth.CONFIGS[2]
    model = synth.make_model(cfg)
    N = 1000
    inp = synth.make_inputs(cfg, N=N, P=8, Q=1, H=1)
    w = np.full(N, 1.0 / N, np.float32)
    parts = inp.bu_particles.copy()
    if bad == "nan_state":
        parts[617, 3] = np.nan
    else:
        w[617] = np.inf
    g = _gpu_bu(torch_cuda, model, parts, 1, inp.observation, w, 5, prec)
    om = oracle.OracleModel(model)
    o = om.belief_update(synth.bf16_round_np(parts) if prec == synth.PREC_BF16 else parts, 1, inp.observation, w, 5)
    assert o["status"] != 0
    assert int(g["status"][0]) == 1
    assert np.array_equal(g["ancestors"], np.arange(N)) and np.array_equal(o["ancestors"], np.arange(N))
    assert np.array_equal(g["particles"], g["proposals"], equal_nan=True)
    if bad == "nan_state":   # the NaN poisons its own row only
        assert np.all(np.isnan(g["proposals"][617])) or np.isnan(g["proposals"][617]).any()
        assert np.isfinite(np.delete(g["proposals"], 617, axis=0)).all()
    assert np.all(g["weights"] == np.float32(1.0) / np.float32(N))
    assert np.isneginf(g["log_evidence"][0]) and np.isneginf(o["log_evidence"])
    # a NaN prior WEIGHT is not > 0: a zero weight on both sides, the update stays regular
    w[617] = np.nan
    g = _gpu_bu(torch_cuda, model, inp.bu_particles, 1, inp.observation, w, 5, prec)
    assert int(g["status"][0]) == 0 and not np.any(g["ancestors"] == 617)


@pytest.fixture(scope="module")
def resample_ctx(torch_cuda):
    import paper_2606_19729_b200 as vl
    ctx = vl.Voila(synth.make_model(synth.CONFIGS[1]))
    yield ctx
    ctx.close()


def _weights_case(kind, N, rng):
    if kind == "skew":      # config 4: log-weights ~ N(0, 4)
        lw = 2.0 * rng.standard_normal(N)
        return np.exp(lw - lw.max()).astype(np.float32)
    if kind == "uniform":
        return np.full(N, 0.37, np.float32)
    if kind == "onehot":
        v = np.zeros(N, np.float32)
        v[N // 3] = 1.0
        return v
    if kind == "sparse":
        v = np.zeros(N, np.float32)
        idx = rng.choice(N, max(1, N // 50), replace=False)
        v[idx] = rng.uniform(0, 1, idx.size).astype(np.float32)
        return v
    if kind == "tiny":      # many weights below 2^-32 (quantise to zero)
        return np.exp(-rng.uniform(0, 40, N)).astype(np.float32)
    raise ValueError(kind)


@pytest.mark.parametrize("N", [1, 2, 31, 256, 2047, 2048, 2049, 100_000, 1_000_000, 1 << 20])
@pytest.mark.parametrize("kind", ["skew", "uniform", "onehot", "sparse", "tiny"])
def test_resample_indices_bit_exact(torch_cuda, oracle, resample_ctx, N, kind):
    """voila_resample_systematic == the oracle's exact-integer definition, for every index."""
    torch = torch_cuda
    rng = np.random.default_rng(N + len(kind))
    v = _weights_case(kind, N, rng)
    ctx = resample_ctx
    for seed in (0, 0xDEADBEEFCAFE):
        anc, status = ctx.voila_resample_systematic(torch.from_numpy(v).cuda(), seed)
        ref, st = oracle.resample_systematic(v, seed)
        # every weight below 2^-32 quantises to zero: both sides flag it and return the identity
        assert int(status.item()) == (0 if st == 0 else 1)
        assert np.array_equal(anc.cpu().numpy(), ref)
        if kind == "uniform":
            assert np.array_equal(ref, np.arange(N))


def test_resample_all_zero(torch_cuda):
    import paper_2606_19729_b200 as vl
    ctx = vl.Voila(synth.make_model(synth.CONFIGS[1]))
    anc, status = ctx.voila_resample_systematic(torch_cuda.zeros(5000, device="cuda"), 9)
    assert int(status.item()) == 1
    assert np.array_equal(anc.cpu().numpy(), np.arange(5000))
    ctx.close()


@pytest.mark.parametrize("cfg_idx", [1, 2, 3])
def test_mlp_forward_fp32(torch_cuda, oracle, cfg_idx):
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg, prec=synth.PREC_FP32)
    ctx = vl.Voila(model, prec=synth.PREC_FP32)
    om = oracle.OracleModel(model)
    rng = np.random.default_rng(cfg_idx)
    for which, f in enumerate(model.mlps()):
        x = rng.standard_normal((77, f.dims[0])).astype(np.float32)
        y = ctx.voila_mlp_forward(which, torch.from_numpy(x).cuda())
        assert_close(t2n(y), om.mlp_forward(which, x), TOL_FP32, f"mlp {which}")
    ctx.close()


def test_belief_update_host_entry(torch_cuda, oracle):
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[2]
    model = synth.make_model(cfg, prec=synth.PREC_FP32)
    inp = synth.make_inputs(cfg, N=3000, P=8, Q=1, H=1)
    dev = _gpu_bu(torch, model, inp.bu_particles, 2, inp.observation, None, 8, synth.PREC_FP32)
    ctx = vl.Voila(model, prec=synth.PREC_FP32)
    parts = torch.from_numpy(inp.bu_particles).pin_memory()
    obs = torch.from_numpy(inp.observation).pin_memory()
    pout = torch.empty_like(parts).pin_memory()
    anc = torch.empty(3000, dtype=torch.int32).pin_memory()
    le = torch.empty(1, dtype=torch.float32).pin_memory()
    st = torch.empty(1, dtype=torch.int32).pin_memory()
    ctx.voila_belief_update_host(parts, 2, obs, None, 8, pout, None, anc, le, st)
    assert int(st.item()) == 0
    assert np.array_equal(anc.numpy(), dev["ancestors"])
    assert np.array_equal(pout.numpy(), dev["particles"])
    ctx.close()


@pytest.mark.parametrize("prec_name,cfg_idx,N", [("fp32", 2, 3000), ("bf16", 3, 5000), ("bf16", 4, 40_001)])
def test_belief_update_adaptive_resampling(torch_cuda, oracle, prec_name, cfg_idx, N):
    """voila_belief_update_ess: ESS against the oracle, both branches of the decision."""
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    bf16 = prec_name == "bf16"
    prec = synth.PREC_BF16 if bf16 else synth.PREC_FP32
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg, prec=prec, lam=1.25)
    inp = synth.make_inputs(cfg, N=N, P=8, Q=1, H=1)
    om = oracle.OracleModel(model)
    src = synth.bf16_round_np(inp.bu_particles) if bf16 else inp.bu_particles
    ref_plain = om.belief_update(src, 1, inp.observation, inp.bu_weights, 77)
    ess_ref = oracle.effective_sample_size(ref_plain["post_weights"])
    ctx = vl.Voila(model, device=0, prec=prec)
    parts = ctx.to_particles(inp.bu_particles)
    obs = torch.from_numpy(inp.observation).cuda()
    w = None if inp.bu_weights is None else torch.from_numpy(inp.bu_weights).cuda()
    frac = ess_ref / N
    for thr, expect in [(2.0 * frac + 0.01, 1), (0.4 * frac, 0)]:  # well away from the boundary (thr may exceed 1)
        out = ctx.voila_belief_update(parts, 1, obs, w, 77, ess_threshold=thr)
        torch.cuda.synchronize()
        g = {k: t2n(v) if v.dtype != torch.int32 else v.cpu().numpy() for k, v in out.items()}
        o = om.belief_update(src, 1, inp.observation, inp.bu_weights, 77, ess_threshold=thr)
        assert int(g["status"][0]) == 0 and o["status"] == 0
        assert int(g["resampled"][0]) == expect == o["resampled"]
        # ESS is a ratio of sums of v_i: a few % in bf16 mode (v_i themselves are within 5e-2)
        assert abs(float(g["ess"][0]) - o["ess"]) <= (0.15 if bf16 else 1e-3) * o["ess"]
        own_ess = oracle.effective_sample_size(g["post_weights"])
        assert abs(float(g["ess"][0]) - own_ess) <= 1e-4 * own_ess     # consistent with its own weights
        if expect:
            anc_ref, st = oracle.resample_systematic(g["post_weights"], 77)
            assert st == 0 and np.array_equal(g["ancestors"], anc_ref)
            assert np.all(g["weights"] == np.float32(1.0) / np.float32(N))
        else:
            assert np.array_equal(g["ancestors"], np.arange(N))
            assert np.array_equal(g["particles"], g["proposals"])
            v = g["post_weights"].astype(np.float64)
            assert np.allclose(g["weights"], v / v.sum(), rtol=2e-6, atol=0)
            assert rel_inf(g["weights"], o["weights"]) <= (5e-2 if bf16 else 2e-4)
    ctx.close()


def test_belief_update_ess_argument_errors(torch_cuda):
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[1]
    ctx = vl.Voila(synth.make_model(cfg))
    inp = synth.make_inputs(cfg, N=64, P=8, Q=1, H=1)
    parts = ctx.to_particles(inp.bu_particles)
    obs = torch.from_numpy(inp.observation).cuda()
    for bad in (0.0, -1.0, float("nan")):
        with pytest.raises(vl.VoilaError):
            ctx.voila_belief_update(parts, 1, obs, None, 1, ess_threshold=bad)
    ctx.close()
