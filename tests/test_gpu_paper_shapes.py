"""GPU parity on PAPER-SHAPED dimensions: TargetFinding has S = R^45, O = R^36 and six actions
(PAPER.md:171-173), LeggedNavigation S = R^39: widths that are not multiples of 8 / 64.
The CTA-pair tcgen05 programs pad them when the weights are packed (public buffers keep their widths);
these tests assert that the tensor-core kernels ran and that the outputs match the oracle."""
import dataclasses

import numpy as np
import pytest

from paper_2606_19729_b200 import synth
from tests.parity_util import TOL_BF16_STATE, TOL_BF16_VALUE, assert_close, t2n, value_err

pytestmark = pytest.mark.gpu


def _cfg(S, O, A, Nz, hidden, tower_hidden, tower_d):
    return dataclasses.replace(synth.CONFIGS[3], name=f"paper_shaped_S{S}", S=S, O=O, A=A, Nz=Nz, hidden=hidden,
                               tower_hidden=tower_hidden, tower_d=tower_d)


@pytest.mark.parametrize("S,O,A,Nz,hidden,reward,P,Q", [
    (39, 36, 6, 12, [200, 200, 200], synth.R_NEG_QUADRATIC, 700, 10),   # LeggedNavigation-sized state, lidar-sized observation
    (45, 36, 6, 5, [200, 136], synth.R_NEG_L2_GOAL, 700, 10),           # TargetFinding-sized state, odd noise width
    (39, 36, 6, 12, [200, 200, 200], synth.R_NEG_QUADRATIC, 1000, 40),  # four blocks x 40 sequences: the two-slot rollout
    (45, 36, 6, 5, [200, 136], synth.R_NEG_L2_GOAL, 400, 80),           # two blocks (the second ragged) x 80 sequences
])
def test_paper_shaped_rollout_and_belief_update(oracle, S, O, A, Nz, hidden, reward, P, Q):
    import torch
    import paper_2606_19729_b200 as vl
    assert torch.cuda.is_available()
    cfg = dataclasses.replace(_cfg(S, O, A, Nz, hidden, [200], 100), reward_kind=reward)
    model = synth.make_model(cfg, action_cost=True)
    H, N = 7, 1500
    inp = synth.make_inputs(cfg, P=P, Q=Q, H=H, N=N)
    ctx = vl.Voila(model, device=0)
    out = ctx.voila_rollout_values(ctx.to_particles(inp.particles), torch.from_numpy(inp.action_seqs).cuda(), None, 77,
                                   want_witness=True, want_returns=True, want_final_states=True)
    w = np.random.default_rng(3).uniform(0.1, 1.0, N).astype(np.float32)
    bu = ctx.voila_belief_update(ctx.to_particles(inp.bu_particles), 2, torch.from_numpy(inp.observation).cuda(),
                                 torch.from_numpy(w).cuda(), 78)
    torch.cuda.synchronize()
    assert "rollout_tc2" in ctx.voila_last_rollout_kernel(), ctx.voila_last_rollout_kernel()
    if Q >= 40:
        assert "rollout_tc2d" in ctx.voila_last_rollout_kernel(), ctx.voila_last_rollout_kernel()
    assert "belief_tc2" in ctx.voila_last_belief_kernel(), ctx.voila_last_belief_kernel()
    om = oracle.OracleModel(model)
    parts = synth.bf16_round_np(inp.particles)
    V, Wit, G = om.rollout_values(parts, inp.action_seqs, None, 77, want_returns=True)
    assert_close(t2n(out["returns"]), G, TOL_BF16_STATE, "returns")
    assert_close(t2n(out["witness"]), Wit, TOL_BF16_STATE, "witness")
    assert value_err(t2n(out["values"]), V) <= TOL_BF16_VALUE
    fin = np.stack([om.rollout_trajectory(parts[p], inp.action_seqs[1], p, 1, 77)[1][H] for p in range(0, P, 7)])
    assert t2n(out["final_states"]).shape == (Q, P, S)
    assert_close(t2n(out["final_states"])[1, ::7], fin, TOL_BF16_STATE, "final states")
    ref = om.belief_update(synth.bf16_round_np(inp.bu_particles), 2, inp.observation, w, 78)
    assert t2n(bu["proposals"]).shape == (N, S)
    assert_close(t2n(bu["proposals"]), ref["proposals"], TOL_BF16_STATE, "proposals")
    assert np.abs(t2n(bu["post_weights"]) - ref["post_weights"]).max() <= 5e-2
    anc_ref, st = oracle.resample_systematic(t2n(bu["post_weights"]), 78)
    anc = bu["ancestors"].cpu().numpy()
    assert st == 0 and np.array_equal(anc, anc_ref)
    assert np.array_equal(t2n(bu["particles"]), t2n(bu["proposals"])[anc])
    ctx.close()
