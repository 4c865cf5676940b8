"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (AUTO kernel,
bf16 mode for CFG2-5): sampled outputs the oracle can compute one by one (a (particle, sequence)
return is one `rollout_trajectory`, keyed by absolute indices), plus properties that hold at any
size.  CFG4's belief update (2^20 particles) is compared in full.  Run on the B200: pytest -m gpu."""
import numpy as np
import pytest

from paper_2606_19729_b200 import synth
from tests.parity_util import TOL_BF16_STATE, TOL_BF16_VALUE, TOL_FP32, rel_inf, t2n

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _sample_pairs(P, Q, n, rng, n_clusters=74):
    """Corners, then pairs spread over the work units of every CTA pair: unit = q * ceil(P/256) + block,
    units go round-robin over the CTA pairs, so the first and the last unit of each pair are hit."""
    pairs = {(0, 0), (P - 1, Q - 1), (P - 1, 0), (0, Q - 1), (P // 2 + 1, Q // 2 - 1)}
    bpq = (P + 255) // 256
    n_units = bpq * Q
    for c in range(min(n_clusters, n_units)):
        last = c + ((n_units - 1 - c) // n_clusters) * n_clusters
        for unit in (c, last):
            q, blk = divmod(unit, bpq)
            p = min(P - 1, blk * 256 + int(rng.integers(256)))
            if len(pairs) < n:
                pairs.add((p, q))
    while len(pairs) < n:
        pairs.add((int(rng.integers(P)), int(rng.integers(Q))))
    return sorted(pairs)


@pytest.mark.parametrize("cfg_idx,n_pairs", [(1, 64), (2, 96), (3, 160), (5, 256)])
def test_rollout_full_size_sampled(torch_cuda, oracle, cfg_idx, n_pairs):
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg)
    bf16 = model.prec == synth.PREC_BF16
    inp = synth.make_inputs(cfg)
    P, (Q, H) = inp.particles.shape[0], inp.action_seqs.shape
    assert (P, Q, H) == (cfg.P, cfg.Q, cfg.H)
    ctx = vl.Voila(model, device=0)
    ctx.voila_reserve(P, Q, H, 16)
    parts = ctx.to_particles(inp.particles)
    seqs = torch.from_numpy(inp.action_seqs).cuda()
    seed = 20260619 + cfg_idx
    out = ctx.voila_rollout_values(parts, seqs, None, seed, want_witness=True, want_returns=True)
    torch.cuda.synchronize()
    kernel = ctx.voila_last_rollout_kernel()
    if bf16:
        assert "rollout_tc2" in kernel, kernel  # what bench.py times
    values, returns, witness = t2n(out["values"]), t2n(out["returns"]), t2n(out["witness"])
    ctx.close()
    assert returns.shape == (Q, P) and np.all(np.isfinite(returns)) and np.all(np.isfinite(witness))

    # (a) sampled returns and discounted observation sums, one oracle trajectory each
    om = oracle.OracleModel(model)
    src = synth.bf16_round_np(inp.particles) if bf16 else inp.particles
    rng = np.random.default_rng(cfg_idx)
    pairs = _sample_pairs(P, Q, n_pairs, rng)
    g_ref = np.array([om.rollout_trajectory(src[p], inp.action_seqs[q], p, q, seed)[0] for p, q in pairs])
    g_gpu = np.array([returns[q, p] for p, q in pairs], np.float64)
    scale = max(float(np.mean(np.abs(g_ref))), 1e-6)
    tol = TOL_BF16_STATE if bf16 else TOL_FP32
    assert np.max(np.abs(g_gpu - g_ref) / np.maximum(np.abs(g_ref), scale)) <= tol

    # (b) any size: V_q is the (uniform-weight) mean of the GPU's own returns; fixed-order double sums
    v_ref = returns.astype(np.float64).mean(axis=1)
    assert np.max(np.abs(values - v_ref)) <= 2e-6 * max(1.0, float(np.max(np.abs(v_ref))))

    # (c) one whole sequence against the oracle (all P particles): value and witness
    q0 = Q - 1
    V, Wit = om.rollout_values(src, inp.action_seqs[q0:q0 + 1], None, seed, q_offset=q0)
    vtol = TOL_BF16_VALUE if bf16 else TOL_FP32
    assert abs(values[q0] - V[0]) <= vtol * max(abs(float(V[0])), float(np.mean(np.abs(values))))
    assert rel_inf(witness[q0], Wit[0]) <= tol


def test_belief_update_full_size_cfg4(torch_cuda, oracle):
    """CFG4 in full: 2^20 particles, heavy weight skew, bf16, the tensor-core propose+score program."""
    import paper_2606_19729_b200 as vl
    from tests.test_gpu_belief import _check_bu
    torch = torch_cuda
    cfg = synth.CONFIGS[4]
    model = synth.make_model(cfg)
    inp = synth.make_inputs(cfg, P=8, Q=1, H=1)
    N = inp.bu_particles.shape[0]
    assert N == 1 << 20 and inp.bu_weights is not None
    ctx = vl.Voila(model, device=0)
    ctx.voila_reserve(8, 1, 1, N)
    parts = ctx.to_particles(inp.bu_particles)
    out = ctx.voila_belief_update(parts, 1, torch.from_numpy(inp.observation).cuda(),
                                  torch.from_numpy(inp.bu_weights).cuda(), 4242)
    torch.cuda.synchronize()
    assert ctx.voila_last_belief_kernel().startswith("belief_tc2_")
    g = {k: t2n(v) if v.dtype != torch.int32 else v.cpu().numpy() for k, v in out.items()}
    ctx.close()
    mism = _check_bu(oracle, model, inp.bu_particles, 1, inp.observation, inp.bu_weights, 4242, g,
                     TOL_BF16_STATE, True)
    # CFG4's skew: effective sample size ~2 %, roughly a third of the proposals survive
    uniq = np.unique(g["ancestors"]).size / N
    assert 0.05 < uniq < 0.6
    print(f"cfg4 full size: end-to-end ancestor mismatch {mism:.4f}, unique ancestors {uniq:.3f}")  # reported only


def test_belief_update_ragged_million(torch_cuda, oracle):
    """N = 10^6 (not a multiple of any tile): properties + bit-exact resampling of the GPU's weights."""
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[4]
    model = synth.make_model(cfg)
    N = 1_000_000
    inp = synth.make_inputs(cfg, P=8, Q=1, H=1, N=N)
    ctx = vl.Voila(model, device=0)
    ctx.voila_reserve(8, 1, 1, N)
    parts = ctx.to_particles(inp.bu_particles)
    w = None if inp.bu_weights is None else torch.from_numpy(inp.bu_weights).cuda()
    out = ctx.voila_belief_update(parts, 2, torch.from_numpy(inp.observation).cuda(), w, 7)
    torch.cuda.synchronize()
    g = {k: t2n(v) if v.dtype != torch.int32 else v.cpu().numpy() for k, v in out.items()}
    ctx.close()
    assert int(g["status"][0]) == 0
    anc_ref, st = oracle.resample_systematic(g["post_weights"], 7)
    assert st == 0 and np.array_equal(g["ancestors"], anc_ref)
    assert np.array_equal(g["particles"], g["proposals"][g["ancestors"]])
    # a prefix of the particles through the oracle (per-particle work is keyed by absolute index)
    M = 4096
    om = oracle.OracleModel(model)
    o = om.belief_update(synth.bf16_round_np(inp.bu_particles[:M]), 2, inp.observation,
                         None if inp.bu_weights is None else inp.bu_weights[:M], 7)
    assert rel_inf(g["proposals"][:M], o["proposals"]) <= TOL_BF16_STATE
