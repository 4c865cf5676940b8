"""GPU property test: the tensor-core kernels (tcgen05 pair path: rollout_tc2x / belief_tc2*) and the
CUDA-core bf16 kernels are independent implementations of the same arithmetic (bf16 operands, fp32
accumulate, the same Philox noise); on seeded random shapes they must agree far inside the bf16
tolerances.  Random P / Q / H / N (ragged tiles, several units per CTA pair, both belief programs)
exercise the event / slot scheduling of the persistent kernels: a scheduling hazard shows up here as
an error of a few per cent.  The oracle parity proper is in test_gpu_rollout.py / test_gpu_belief.py."""
import numpy as np
import pytest

from paper_2606_19729_b200 import synth

pytestmark = pytest.mark.gpu


def _rel_l2(a, b):
    a, b = a.double(), b.double()
    return float((a - b).norm() / max(float(b.norm()), 1e-30))


@pytest.mark.parametrize("cfg_idx", [2, 3, 4, 5])
def test_tensor_core_and_cuda_core_kernels_agree(cfg_idx):
    import torch
    import paper_2606_19729_b200 as vl
    assert torch.cuda.is_available()
    rng = np.random.default_rng(1000 + cfg_idx)
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg, prec=synth.PREC_BF16, lik_action_cond=cfg_idx % 2)
    ctx = vl.Voila(model, device=0, prec=synth.PREC_BF16)
    if not ctx.voila_tcgen05_supported():
        ctx.close()
        pytest.skip("tcgen05 path does not support these dims")
    for trial in range(10):
        P, Q, H = int(rng.integers(1, 5000)), int(rng.integers(1, 40)), int(rng.integers(1, 9))
        N = int(rng.integers(1, 3000)) if trial % 2 else int(rng.integers(19_000, 60_000))
        inp = synth.make_inputs(cfg, P=P, Q=Q, H=H, N=N, seed=int(rng.integers(1 << 30)))
        parts, bup = ctx.to_particles(inp.particles), ctx.to_particles(inp.bu_particles)
        seqs = torch.from_numpy(inp.action_seqs).cuda()
        w = torch.from_numpy(np.exp(rng.standard_normal(P)).astype(np.float32)).cuda() if trial % 3 else None
        bw = None if inp.bu_weights is None else torch.from_numpy(inp.bu_weights).cuda()
        obs = torch.from_numpy(inp.observation).cuda()
        seed, action = int(rng.integers(1 << 40)), int(rng.integers(cfg.A))
        res = {}
        for name, kernel in (("tc", vl.KERNEL_TCGEN05_PAIR), ("ffma", vl.KERNEL_FFMA)):
            ctx.voila_set_kernel(kernel)
            out = ctx.voila_rollout_values(parts, seqs, w, seed, want_witness=True, want_returns=True)
            bu = ctx.voila_belief_update(bup, action, obs, bw, seed + 1)
            torch.cuda.synchronize()
            res[name] = (out, bu)
        what = f"cfg{cfg_idx} P={P} Q={Q} H={H} N={N}"
        assert _rel_l2(res["tc"][0]["returns"], res["ffma"][0]["returns"]) <= 5e-3, what
        assert _rel_l2(res["tc"][0]["witness"], res["ffma"][0]["witness"]) <= 5e-3, what
        assert _rel_l2(res["tc"][1]["proposals"].float(), res["ffma"][1]["proposals"].float()) <= 5e-3, what
        assert float((res["tc"][1]["post_weights"] - res["ffma"][1]["post_weights"]).abs().max()) <= 2e-2, what
    ctx.close()


@pytest.mark.parametrize("cfg_idx", [2, 3, 4])
def test_two_slot_rollout_and_cuda_core_kernels_agree(cfg_idx):
    """The two-slot rollout kernel (rollout_tc2d_kernel: two 256-particle blocks of a sequence in flight
    per CTA pair) against the CUDA-core bf16 kernel on random shapes that select it: an even number of
    256-particle blocks (the last one ragged), more pairs of blocks than CTA pairs, several units per
    CTA pair, with and without prior weights."""
    import torch
    import paper_2606_19729_b200 as vl
    assert torch.cuda.is_available()
    rng = np.random.default_rng(2000 + cfg_idx)
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg, prec=synth.PREC_BF16)
    ctx = vl.Voila(model, device=0, prec=synth.PREC_BF16)
    for trial in range(8):
        pairs = int(rng.integers(1, 5))                                # pairs of 256-particle blocks per sequence
        P = 512 * pairs - int(rng.integers(0, 256))                    # ragged last block, block count stays even
        Q = int(rng.integers(75 // pairs + 1, 75 // pairs + 60))       # pairs * Q > 74 CTA pairs
        H = int(rng.integers(1, 7))
        inp = synth.make_inputs(cfg, P=P, Q=Q, H=H, N=8, seed=int(rng.integers(1 << 30)))
        parts = ctx.to_particles(inp.particles)
        seqs = torch.from_numpy(inp.action_seqs).cuda()
        w = torch.from_numpy(np.exp(rng.standard_normal(P)).astype(np.float32)).cuda() if trial % 2 else None
        seed = int(rng.integers(1 << 40))
        res = {}
        for name, kernel in (("tc", vl.KERNEL_AUTO), ("ffma", vl.KERNEL_FFMA)):
            ctx.voila_set_kernel(kernel)
            res[name] = ctx.voila_rollout_values(parts, seqs, w, seed, want_witness=True, want_returns=True,
                                                 want_final_states=True)
            torch.cuda.synchronize()
            if name == "tc":
                assert "rollout_tc2d_kernel" in ctx.voila_last_rollout_kernel(), ctx.voila_last_rollout_kernel()
        what = f"cfg{cfg_idx} P={P} Q={Q} H={H}"
        assert _rel_l2(res["tc"]["returns"], res["ffma"]["returns"]) <= 5e-3, what
        assert _rel_l2(res["tc"]["witness"], res["ffma"]["witness"]) <= 5e-3, what
        assert _rel_l2(res["tc"]["final_states"].float(), res["ffma"]["final_states"].float()) <= 5e-3, what
        assert _rel_l2(res["tc"]["values"], res["ffma"]["values"]) <= 5e-3, what
    ctx.close()
