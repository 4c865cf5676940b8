"""GPU parity of the CHAINED planning loop bench.py times (config-5 protocol): rollout ->
executed action = first action of argmax_q V -> belief update on the observation -> rollout on the
resampled particles ...  At every step the oracle is fed the GPU's own particles and chosen action
(SURVEY 8c O7 extended to states), so steps 2 and 3 are checked element by element too, not only step 1.
Also: out-of-range actions are clamped by the kernels."""
import numpy as np
import pytest

from paper_2606_19729_b200 import synth
from tests.parity_util import TOL_BF16_STATE, TOL_BF16_VALUE, assert_close, t2n, value_err

pytestmark = pytest.mark.gpu


def test_cfg5_protocol_three_chained_steps(oracle):
    import torch
    import paper_2606_19729_b200 as vl
    assert torch.cuda.is_available()
    cfg = synth.CONFIGS[5]
    model = synth.make_model(cfg)
    P, Q, H, steps = 768, 12, 6, 3  # the config-5 model and protocol on a slice the oracle finishes in seconds
    inp = synth.make_inputs(cfg, P=P, Q=Q, H=H, N=P)
    obs = synth.observations_for_steps(cfg, steps)
    ctx = vl.Voila(model, device=0)
    om = oracle.OracleModel(model)
    parts = ctx.to_particles(inp.particles)
    seqs = torch.from_numpy(inp.action_seqs).cuda()
    for k in range(steps):
        out = ctx.voila_rollout_values(parts, seqs, None, 100 + 2 * k, want_witness=True, want_returns=True)
        bq, ba = ctx.voila_best_action(out["values"], seqs)
        a_exec = int(ba.item())
        bu = ctx.voila_belief_update(parts, a_exec, torch.from_numpy(obs[k]).cuda(), None, 101 + 2 * k)
        torch.cuda.synchronize()
        assert "rollout_tc2" in ctx.voila_last_rollout_kernel() and "belief_tc2" in ctx.voila_last_belief_kernel()
        parts_np = t2n(parts)  # the GPU's own particles of this step (bf16 values)
        # planning half
        V, Wit, G = om.rollout_values(parts_np, inp.action_seqs, None, 100 + 2 * k, want_returns=True)
        assert_close(t2n(out["returns"]), G, TOL_BF16_STATE, f"step {k} returns")
        assert_close(t2n(out["witness"]), Wit, TOL_BF16_STATE, f"step {k} witness")
        assert value_err(t2n(out["values"]), V) <= TOL_BF16_VALUE
        vg = t2n(out["values"])
        assert int(bq.item()) == int(np.argmax(vg)) and a_exec == int(inp.action_seqs[int(np.argmax(vg)), 0])
        # filtering half, with the action the GPU executed
        ref = om.belief_update(parts_np, a_exec, obs[k], None, 101 + 2 * k)
        assert_close(t2n(bu["proposals"]), ref["proposals"], TOL_BF16_STATE, f"step {k} proposals")
        assert np.abs(t2n(bu["post_weights"]) - ref["post_weights"]).max() <= 5e-2
        anc_ref, st = oracle.resample_systematic(t2n(bu["post_weights"]), 101 + 2 * k)
        anc = bu["ancestors"].cpu().numpy()
        assert st == 0 and np.array_equal(anc, anc_ref)
        assert np.array_equal(t2n(bu["particles"]), t2n(bu["proposals"])[anc])
        parts = bu["particles"]  # the next step plans from the resampled belief
    ctx.close()


@pytest.mark.parametrize("prec", [synth.PREC_FP32, synth.PREC_BF16])
def test_out_of_range_actions_are_clamped(prec):
    import torch
    import paper_2606_19729_b200 as vl
    cfg = synth.CONFIGS[2]
    model = synth.make_model(cfg, prec=prec, action_cost=True)
    inp = synth.make_inputs(cfg, P=300, Q=6, H=5)
    ctx = vl.Voila(model, device=0, prec=prec)
    parts = ctx.to_particles(inp.particles)
    good = inp.action_seqs.copy()
    good[1, :] = cfg.A - 1
    good[2, 3] = 0
    bad = good.copy()
    bad[1, :] = cfg.A + 7
    bad[2, 3] = -4
    res = []
    for s in (good, bad):
        out = ctx.voila_rollout_values(parts, torch.from_numpy(s).cuda(), None, 9, want_returns=True)
        torch.cuda.synchronize()
        res.append({k: t2n(v) for k, v in out.items()})
    for k in res[0]:
        assert np.array_equal(res[0][k], res[1][k]), k
    ctx.close()
