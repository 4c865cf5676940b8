"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (AUTO kernel,
bf16 mode for CFG2-5): sampled outputs the oracle can compute one by one (a (particle, sequence)
return is one `rollout_trajectory`, keyed by absolute indices), plus properties that hold at any
size.  CFG4's belief update (2^20 particles) is compared in full.  Run on the B200: pytest -m gpu."""
import numpy as np
import pytest

from paper_2606_19729_b200 import synth
from tests.parity_util import TOL_BF16_STATE, TOL_BF16_VALUE, TOL_FP32, rel_inf, rel_l2, t2n

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
        # ... in the launch configuration it times: the two-slot kernel for the <= 256-wide generators
        # (configs 2, 3), the 16-epilogue-warp one-block kernel for config 5
        assert ("rollout_tc2d_kernel" if cfg_idx in (2, 3) else "rollout_tc2x_kernel") in kernel, kernel
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


def test_progressive_widening_bench_size(torch_cuda, oracle):
    """The progressive-widening leg of bench.py (2^18 simulations, 2048 ragged action nodes, M_max = 16,
    config-3 model, two-slot tcgen05 program): every integer output against the oracle, ancestors bit-exact
    given the GPU's own weights child by child, proposals on a sample of rows."""
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[3]
    model = synth.make_model(cfg)
    N, G, M = 1 << 18, 2048, 16
    rng = np.random.default_rng(20260619 + 77)
    parts = rng.standard_normal((N, cfg.S)).astype(np.float32)
    cuts = np.concatenate([[0], np.sort(rng.integers(0, N + 1, G - 1)), [N]]).astype(np.int32)
    acts = rng.integers(0, cfg.A, G).astype(np.int32)
    bc0 = rng.integers(0, M // 2 + 1, G).astype(np.int32)
    vc0 = (bc0 * 8).astype(np.int32)
    bo0 = rng.standard_normal((G, M, cfg.O)).astype(np.float32)
    ctx = vl.Voila(model, device=0)
    t = lambda a: torch.from_numpy(a.copy()).cuda()
    t_vc, t_bc, t_bo = t(vc0), t(bc0), t(bo0)
    out = ctx.voila_pw_update(ctx.to_particles(parts), t(cuts), t(acts), t_vc, t_bc, t_bo, 1.5, 0.5, None, 9000)
    torch.cuda.synchronize()
    assert "belief_tc2_dual_kernel" in ctx.voila_last_belief_kernel()
    g = {k: (t2n(v) if v.dtype.is_floating_point else v.cpu().numpy()) for k, v in out.items()}
    ctx.close()
    ref = oracle.OracleModel(model, emulate_bf16=True).pw_update(synth.bf16_round_np(parts), cuts, acts, vc0, bc0, bo0,
                                                                  1.5, 0.5, None, 9000)
    for k in ("sim_branch", "opened", "seg_status"):
        assert np.array_equal(g[k], ref[k]), k
    assert np.array_equal(t_bc.cpu().numpy(), ref["branch_count"]) and np.array_equal(t_vc.cpu().numpy(), ref["visit_count"])
    rows = rng.choice(N, 4096, replace=False)
    assert rel_inf(g["proposals"][rows], ref["proposals"][rows]) <= TOL_BF16_STATE
    opened = np.flatnonzero(ref["opened"])[:512]
    gb, rb = t_bo.cpu().numpy(), ref["branch_obs"]
    for i in opened:
        gi = int(np.searchsorted(cuts, i, side="right") - 1)
        b = int(ref["sim_branch"][i])
        assert np.abs(gb[gi, b] - rb[gi, b]).max() <= 2 * TOL_BF16_STATE * max(1.0, float(np.abs(rb[gi, b]).max()))
    # children: resampled among their own members, bit-exact given the GPU's weights (a sample of nodes)
    seg = np.repeat(np.arange(G), np.diff(cuts)) * M + ref["sim_branch"]
    for gi in rng.choice(G, 64, replace=False):
        idx = np.arange(cuts[gi], cuts[gi + 1])
        for b in range(ref["branch_count"][gi]):
            mem = idx[ref["sim_branch"][idx] == b]
            if mem.size == 0:
                continue
            v = g["post_weights"][mem]
            x0 = oracle.philox4x32_10([gi * M + b, 0, 0, 4 << 16], [9000, 0])[0]
            a_loc, st = oracle.resample_systematic_x0(v, int(x0))
            assert st == 0 and np.array_equal(g["ancestors"][mem], mem[a_loc])
    assert np.array_equal(seg[g["ancestors"]], seg)  # every draw stays inside its child, for ALL simulations
    assert np.array_equal(g["particles"], g["proposals"][g["ancestors"]])


def test_diffusion_teacher_bench_size_sampled(torch_cuda, oracle):
    """The diffusion-teacher leg of bench.py (2^16 samples, 4 x 512 denoiser, K = 32): the first 1024 samples
    against the oracle (the noise is keyed by the absolute sample index, so a prefix reproduces them)."""
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[3]
    vT, vZ = synth.make_denoisers(cfg, [512, 512, 512, 512])
    model = synth.make_model(cfg).replace(denoise_T=vT, denoise_Z=vZ)
    N, K, n_ref = 1 << 16, 32, 1024
    rng = np.random.default_rng(20260619 + 88)
    cond = rng.standard_normal((N, cfg.S)).astype(np.float32)
    act = rng.integers(0, cfg.A, N).astype(np.int32)
    ctx = vl.Voila(model, device=0)
    out = t2n(ctx.voila_diffusion_sample(0, ctx.to_particles(cond), torch.from_numpy(act).cuda(), K, 2))
    torch.cuda.synchronize()
    assert "belief_tc2_kernel" in ctx.voila_last_belief_kernel()
    ctx.close()
    ref = oracle.OracleModel(model, emulate_bf16=True).diffusion_sample(0, synth.bf16_round_np(cond[:n_ref]), act[:n_ref], K, 2)
    assert np.all(np.isfinite(out))
    assert rel_l2(out[:n_ref], ref) <= TOL_BF16_STATE and rel_inf(out[:n_ref], ref) <= TOL_BF16_STATE
