"""GPU parity: voila_pw_update (vectorised progressive widening with batched likelihood, SURVEY 8f f1;
PAPER.md:147-149) through the C ABI against the oracle.  Integer work (widening decisions, branch of
every simulation, counts) is bit-exact; floats within the north-star tolerances; resampled indices
bit-exact given identical weights (the GPU's own v_i go through the oracle's resampler child by child)."""
import numpy as np
import pytest

from paper_2606_19729_b200 import synth
from tests.parity_util import TOL_BF16_STATE, TOL_FP32, assert_close, t2n

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    return torch


def _groups(rng, N, G, A, empty_some=True):
    if G == 1:
        cuts = np.array([0, N], np.int32)
    else:
        inner = np.sort(rng.integers(0, N + 1, G - 1)) if empty_some else np.sort(
            rng.choice(np.arange(1, N), G - 1, replace=False))
        cuts = np.concatenate([[0], inner, [N]]).astype(np.int32)
    return cuts, rng.integers(0, A, G).astype(np.int32)


def _run_case(torch, oracle, cfg_idx, prec, N, G, M_max, k_o, alpha_o, seed, with_weights=True, prefill=True,
              lik_action_cond=0, zero_child=False):
    import paper_2606_19729_b200 as vl
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg, prec=prec, lik_action_cond=lik_action_cond)
    rng = np.random.default_rng(seed)
    bf16 = prec == synth.PREC_BF16
    parts = rng.standard_normal((N, cfg.S)).astype(np.float32)
    parts_np = synth.bf16_round_np(parts) if bf16 else parts
    cuts, acts = _groups(rng, N, G, cfg.A)
    bc0 = rng.integers(0, M_max // 2 + 1, G).astype(np.int32) if prefill else np.zeros(G, np.int32)
    vc0 = (bc0 * 3 + rng.integers(0, 5, G)).astype(np.int32)
    bo0 = rng.standard_normal((G, M_max, cfg.O)).astype(np.float32)
    w = rng.uniform(0.05, 1.0, N).astype(np.float32) if with_weights else None
    om = oracle.OracleModel(model, emulate_bf16=bf16)
    if zero_child:  # kill one child belief: every simulation the oracle attaches to (g0, b0) gets weight 0
        first = om.pw_update(parts_np, cuts, acts, vc0, bc0, bo0, k_o, alpha_o, w, seed)
        g0 = int(np.argmax(np.diff(cuts)))
        idx = np.arange(cuts[g0], cuts[g0 + 1])
        w = w.copy()
        w[idx[first["sim_branch"][idx] == 0]] = 0.0
    ref = om.pw_update(parts_np, cuts, acts, vc0, bc0, bo0, k_o, alpha_o, w, seed)

    ctx = vl.Voila(model, device=0, prec=prec)
    dev = "cuda:0"
    t_vc, t_bc = torch.from_numpy(vc0.copy()).to(dev), torch.from_numpy(bc0.copy()).to(dev)
    t_bo = torch.from_numpy(bo0.copy()).to(dev)
    out = ctx.voila_pw_update(ctx.to_particles(parts), torch.from_numpy(cuts).to(dev), torch.from_numpy(acts).to(dev),
                              t_vc, t_bc, t_bo, k_o, alpha_o, None if w is None else torch.from_numpy(w).to(dev), seed)
    torch.cuda.synchronize()
    g = {k: t2n(v) if v.dtype.is_floating_point else v.cpu().numpy() for k, v in out.items()}
    g["visit_count"], g["branch_count"], g["branch_obs"] = t_vc.cpu().numpy(), t_bc.cpu().numpy(), t_bo.cpu().numpy()
    launches = ctx.voila_launch_count()
    kname = ctx.voila_last_belief_kernel()
    ctx.close()
    assert launches >= 10

    # integer work: bit-exact
    for k in ("sim_branch", "opened", "visit_count", "branch_count", "seg_status"):
        assert np.array_equal(g[k], ref[k]), k
    tol = TOL_BF16_STATE if bf16 else TOL_FP32
    assert_close(g["proposals"], ref["proposals"], tol, "proposals")
    # stored observations: rows of branches opened in this call hold f_Z's sample, the others are untouched
    for gi in range(G):
        for b in range(M_max):
            if bc0[gi] <= b < ref["branch_count"][gi]:
                e = np.abs(g["branch_obs"][gi, b] - ref["branch_obs"][gi, b]).max()
                assert e <= 2 * tol * max(1.0, np.abs(ref["branch_obs"][gi, b]).max()), (gi, b, e)
            else:
                assert np.array_equal(g["branch_obs"][gi, b], bo0[gi, b])
    assert np.abs(g["post_weights"] - ref["post_weights"]).max() <= (5e-2 if bf16 else 2e-4)
    # resampling per child belief: bit-exact given the GPU's own weights
    n_children = 0
    for gi in range(G):
        idx = np.arange(cuts[gi], cuts[gi + 1])
        for b in range(ref["branch_count"][gi]):
            mem = idx[ref["sim_branch"][idx] == b]
            if mem.size == 0:
                continue
            np.testing.assert_allclose(g["weights"][mem], 1.0 / mem.size, rtol=1e-6)
            if ref["seg_status"][gi * M_max + b]:
                assert np.array_equal(g["ancestors"][mem], mem)
                continue
            n_children += 1
            v = g["post_weights"][mem]
            assert v.max() == 1.0
            x0 = oracle.philox4x32_10([gi * M_max + b, 0, 0, 4 << 16], [seed & 0xffffffff, seed >> 32])[0]
            a_loc, st = oracle.resample_systematic_x0(v, int(x0))
            assert st == 0 and np.array_equal(g["ancestors"][mem], mem[a_loc]), (gi, b)
    assert np.array_equal(g["particles"], g["proposals"][g["ancestors"]])
    ref["kernel"] = kname
    return n_children, ref


def test_pw_fp32_ragged_groups(torch_cuda, oracle):
    n, ref = _run_case(torch_cuda, oracle, 1, synth.PREC_FP32, N=700, G=9, M_max=6, k_o=1.3, alpha_o=0.5, seed=41)
    assert n >= 12 and ref["opened"].sum() >= 5


def test_pw_fp32_many_small_groups(torch_cuda, oracle):
    n, _ = _run_case(torch_cuda, oracle, 1, synth.PREC_FP32, N=900, G=260, M_max=4, k_o=1.0, alpha_o=0.7, seed=42)
    assert n >= 200


def test_pw_fp32_one_large_group_from_scratch(torch_cuda, oracle):
    """A single action node visited 5000 times in one batch, starting empty: the widening recursion over
    many warp chunks (k = 2, alpha = 1/2 hits exact squares), M_max reached."""
    n, ref = _run_case(torch_cuda, oracle, 1, synth.PREC_FP32, N=5000, G=1, M_max=64, k_o=2.0, alpha_o=0.5, seed=43,
                       prefill=False, with_weights=False)
    assert ref["branch_count"][0] == 64 and n == 64


@pytest.mark.parametrize("cfg_idx,lac", [(2, 0), (3, 0), (2, 1)])
def test_pw_bf16(torch_cuda, oracle, cfg_idx, lac):
    n, ref = _run_case(torch_cuda, oracle, cfg_idx, synth.PREC_BF16, N=800, G=12, M_max=8, k_o=1.5, alpha_o=0.45,
                       seed=44 + cfg_idx, lik_action_cond=lac)
    assert n >= 20
    # the fused per-row-action tcgen05 program serves the call unless the state tower is action-conditioned
    assert ("belief_tc2_kernel" in ref["kernel"]) == (lac == 0), ref["kernel"]


def test_pw_bf16_two_units_in_flight(torch_cuda, oracle):
    """Enough simulations for the two-slot program (N > 256 x CTA pairs), ragged tail, 40 action nodes."""
    n, ref = _run_case(torch_cuda, oracle, 3, synth.PREC_BF16, N=40001, G=40, M_max=16, k_o=2.0, alpha_o=0.4, seed=50)
    assert n >= 300 and "belief_tc2_dual_kernel" in ref["kernel"], ref["kernel"]


def test_pw_zero_weight_child(torch_cuda, oracle):
    _, ref = _run_case(torch_cuda, oracle, 1, synth.PREC_FP32, N=400, G=3, M_max=5, k_o=1.0, alpha_o=0.5, seed=46,
                       zero_child=True)
    assert ref["seg_status"].sum() >= 1


def test_pw_argument_errors(torch_cuda):
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[1]
    ctx = vl.Voila(synth.make_model(cfg), device=0)
    parts = ctx.to_particles(np.zeros((8, cfg.S), np.float32))
    go = torch.tensor([0, 8], dtype=torch.int32, device="cuda")
    ga = torch.zeros(1, dtype=torch.int32, device="cuda")
    vc, bc = torch.zeros(1, dtype=torch.int32, device="cuda"), torch.zeros(1, dtype=torch.int32, device="cuda")
    bo = torch.zeros((1, 4, cfg.O), device="cuda")
    with pytest.raises(vl.VoilaError):
        ctx.voila_pw_update(parts, go, ga, vc, bc, bo, -1.0, 0.5, None, 1)
    with pytest.raises(vl.VoilaError):
        ctx.voila_pw_update(parts, go, ga, vc, bc, torch.zeros((1, 65, cfg.O), device="cuda"), 1.0, 0.5, None, 1)
    ctx.close()
