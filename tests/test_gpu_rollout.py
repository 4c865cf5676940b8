"""GPU parity: voila_rollout_values (through the C ABI) against the CPU oracle, element by element
on the same seeded inputs.  Run on the B200 box: pytest -m gpu."""
import numpy as np
import pytest

from paper_2606_19729_b200 import synth
from tests.parity_util import (TOL_BF16_STATE, TOL_BF16_VALUE, TOL_FP32, assert_close, rel_l2, t2n,
                               value_err)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _run_gpu(torch, model, inp, prec, kernel, weights=None, seed=1234, want_final=True):
    import paper_2606_19729_b200 as vl
    ctx = vl.Voila(model, device=0, prec=prec)
    if kernel == vl.KERNEL_TCGEN05 and not ctx.voila_tcgen05_supported():
        ctx.close()
        pytest.skip("tcgen05 path does not support these dims")
    ctx.voila_set_kernel(kernel)
    parts = ctx.to_particles(inp.particles)
    seqs = torch.from_numpy(inp.action_seqs).cuda()
    w = None if weights is None else torch.from_numpy(weights).cuda()
    out = ctx.voila_rollout_values(parts, seqs, w, seed, want_witness=True, want_returns=True,
                                   want_final_states=want_final)
    torch.cuda.synchronize()
    res = {k: t2n(v) for k, v in out.items() if v is not None}
    res["kernel"] = ctx.voila_last_rollout_kernel()
    res["launches"] = ctx.voila_launch_count()
    ctx.close()
    return res


def _run_oracle(oracle, model, inp, weights=None, seed=1234, emulate_bf16=False, bf16_inputs=False,
                want_final=True):
    om = oracle.OracleModel(model, emulate_bf16=emulate_bf16)
    parts = synth.bf16_round_np(inp.particles) if bf16_inputs else inp.particles
    V, Wit, G = om.rollout_values(parts, inp.action_seqs, weights, seed, want_returns=True)
    res = {"values": V, "witness": Wit, "returns": G}
    if want_final:
        Q, H = inp.action_seqs.shape
        P = parts.shape[0]
        fin = np.zeros((Q, P, model.S), np.float32)
        for q in range(Q):
            for p in range(P):
                _, states, _ = om.rollout_trajectory(parts[p], inp.action_seqs[q], p, q, seed)
                fin[q, p] = states[H]
        res["final_states"] = fin
    return res


def test_cfg1_fp32_full(torch_cuda, oracle):
    """BASELINE config 1 at full size, fp32 mode: every output within relative 1e-4."""
    import paper_2606_19729_b200 as vl
    cfg = synth.CONFIGS[1]
    model = synth.make_model(cfg, prec=synth.PREC_FP32)
    inp = synth.make_inputs(cfg)
    g = _run_gpu(torch_cuda, model, inp, synth.PREC_FP32, vl.KERNEL_AUTO)
    o = _run_oracle(oracle, model, inp)
    assert g["launches"] >= 3
    assert_close(g["final_states"], o["final_states"], TOL_FP32, "final states")
    assert_close(g["returns"], o["returns"], TOL_FP32, "returns")
    assert_close(g["witness"], o["witness"], TOL_FP32, "witness")
    assert value_err(g["values"], o["values"]) <= TOL_FP32


@pytest.mark.parametrize("P,Q,H", [(200, 24, 15), (1, 1, 1), (33, 3, 2), (257, 5, 7)])
def test_cfg2_fp32_ragged_weighted(torch_cuda, oracle, P, Q, H):
    """Config 2 shapes at sizes spanning several tiles plus a ragged tail, non-uniform prior weights
    (some exactly zero), SiLU generators, fp32 mode."""
    import paper_2606_19729_b200 as vl
    cfg = synth.CONFIGS[2]
    model = synth.make_model(cfg, prec=synth.PREC_FP32, action_cost=True)
    inp = synth.make_inputs(cfg, P=P, Q=Q, H=H)
    rng = np.random.default_rng(5)
    w = rng.uniform(0.0, 2.0, P).astype(np.float32)
    if P > 4:
        w[::7] = 0.0
    g = _run_gpu(torch_cuda, model, inp, synth.PREC_FP32, vl.KERNEL_AUTO, weights=w)
    o = _run_oracle(oracle, model, inp, weights=w)
    assert_close(g["final_states"], o["final_states"], TOL_FP32, "final states")
    assert_close(g["returns"], o["returns"], TOL_FP32, "returns")
    assert_close(g["witness"], o["witness"], TOL_FP32, "witness")
    assert value_err(g["values"], o["values"]) <= TOL_FP32


def test_cfg3_fp32_quadratic_reward(torch_cuda, oracle):
    """Config 3 dims (S=48, O=64, A=16, Nz=16, 3x256) with the quadratic reward, fp32 mode."""
    import paper_2606_19729_b200 as vl
    cfg = synth.CONFIGS[3]
    model = synth.make_model(cfg, prec=synth.PREC_FP32)
    inp = synth.make_inputs(cfg, P=70, Q=3, H=6)
    g = _run_gpu(torch_cuda, model, inp, synth.PREC_FP32, vl.KERNEL_AUTO)
    o = _run_oracle(oracle, model, inp)
    assert_close(g["final_states"], o["final_states"], TOL_FP32, "final states")
    assert_close(g["returns"], o["returns"], TOL_FP32, "returns")
    assert value_err(g["values"], o["values"]) <= TOL_FP32


def test_linear_reward_relu_none(torch_cuda, oracle):
    """Linear generators (act NONE) with the linear reward: the closed-form pin's model on the GPU."""
    import paper_2606_19729_b200 as vl
    rng = np.random.default_rng(11)
    S, O, A, Nz = 3, 2, 4, 2
    gin = S + A + Nz
    f_T = synth.make_mlp(rng, [gin, S], synth.ACT_NONE)
    f_Z = synth.make_mlp(rng, [gin, O], synth.ACT_NONE)
    lo = synth.make_mlp(rng, [O, 4, 3], synth.ACT_NONE)
    ls = synth.make_mlp(rng, [S, 4, 3], synth.ACT_NONE)
    c = rng.standard_normal(S + 1).astype(np.float32)
    model = synth.ModelSpec(S, O, A, Nz, f_T, f_Z, lo, ls, gamma=0.9, reward_kind=synth.R_LINEAR,
                            reward_param=c, action_cost=rng.uniform(-.3, 0, A).astype(np.float32))
    inp = synth.Inputs(rng.standard_normal((37, S)).astype(np.float32),
                       rng.integers(0, A, (6, 7), dtype=np.int32), None, None, None, None, 0, 0)
    g = _run_gpu(torch_cuda, model, inp, synth.PREC_FP32, vl.KERNEL_AUTO)
    o = _run_oracle(oracle, model, inp)
    assert_close(g["returns"], o["returns"], TOL_FP32, "returns")
    assert_close(g["final_states"], o["final_states"], TOL_FP32, "final states")


def _bf16_case(torch, oracle, cfg_idx, P, Q, H, kernel, seed=99, gain=1.0):
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg, prec=synth.PREC_BF16, gain=gain)
    inp = synth.make_inputs(cfg, P=P, Q=Q, H=H)
    g = _run_gpu(torch, model, inp, synth.PREC_BF16, kernel, seed=seed)
    o = _run_oracle(oracle, model, inp, seed=seed, bf16_inputs=True)
    e = _run_oracle(oracle, model, inp, seed=seed, bf16_inputs=True, emulate_bf16=True,
                    want_final=False)
    return g, o, e


@pytest.mark.parametrize("kernel_name", ["ffma", "tcgen05", "tcgen05_pair"])
@pytest.mark.parametrize("cfg_idx,P,Q,H", [(2, 300, 6, 15), (3, 200, 3, 20), (5, 130, 2, 10), (5, 700, 3, 6)])
def test_bf16_mode_within_north_star(torch_cuda, oracle, kernel_name, cfg_idx, P, Q, H):
    """bf16 mode against the fp32 oracle: relative 2e-2 on states, 1e-2 on value estimates."""
    import paper_2606_19729_b200 as vl
    kernel = {"ffma": vl.KERNEL_FFMA, "tcgen05": vl.KERNEL_TCGEN05,
              "tcgen05_pair": vl.KERNEL_TCGEN05_PAIR}[kernel_name]
    g, o, e = _bf16_case(torch_cuda, oracle, cfg_idx, P, Q, H, kernel)
    if kernel_name == "tcgen05":
        assert "rollout_tc_kernel" in g["kernel"], g["kernel"]
    if kernel_name == "tcgen05_pair":
        assert "rollout_tc2" in g["kernel"], g["kernel"]
    assert_close(g["final_states"], o["final_states"], TOL_BF16_STATE, "final states")
    assert value_err(g["values"], o["values"]) <= TOL_BF16_VALUE
    assert value_err(g["returns"], o["returns"]) <= TOL_BF16_STATE
    assert_close(g["witness"], o["witness"], TOL_BF16_STATE, "witness")
    # against the oracle's bf16-emulation hook the gap is rounding-order only
    assert rel_l2(g["returns"], e["returns"]) <= 5e-3


@pytest.mark.parametrize("cfg_idx,P,Q,H,weighted", [(2, 300, 80, 6, False), (3, 1000, 40, 4, True),
                                                    (3, 512, 75, 3, False), (2, 512, 150, 1, True),
                                                    (2, 1200, 30, 3, True)])
def test_bf16_two_slot_rollout(torch_cuda, oracle, cfg_idx, P, Q, H, weighted):
    """Generators <= 256 wide, an even number of 256-particle blocks per sequence (or >= 5: P = 1200 is five
    blocks, the last pair's second slot stays empty) and more pairs of blocks than CTA pairs: AUTO runs the two-slot kernel (two blocks of one sequence in flight per CTA
    pair, one set of stateful epilogue warps each).  Ragged last block, zero weights, every output."""
    import paper_2606_19729_b200 as vl
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg, prec=synth.PREC_BF16, action_cost=True)
    inp = synth.make_inputs(cfg, P=P, Q=Q, H=H)
    w = None
    if weighted:
        w = np.random.default_rng(3).uniform(0.0, 2.0, P).astype(np.float32)
        w[::5] = 0.0
    g = _run_gpu(torch_cuda, model, inp, synth.PREC_BF16, vl.KERNEL_AUTO, weights=w, seed=7)
    assert "rollout_tc2d_kernel" in g["kernel"], g["kernel"]
    o = _run_oracle(oracle, model, inp, weights=w, seed=7, bf16_inputs=True)
    assert_close(g["final_states"], o["final_states"], TOL_BF16_STATE, "final states")
    assert value_err(g["values"], o["values"]) <= TOL_BF16_VALUE
    assert value_err(g["returns"], o["returns"]) <= TOL_BF16_STATE
    assert_close(g["witness"], o["witness"], TOL_BF16_STATE, "witness")
    # same inputs through the one-block kernel family: same arithmetic per row, so the per-trajectory
    # returns agree to rounding order of the tensor-core accumulation (not bit-exact: block shapes differ)
    h = _run_gpu(torch_cuda, model, inp, synth.PREC_BF16, vl.KERNEL_TCGEN05, weights=w, seed=7, want_final=False)
    assert rel_l2(g["returns"], h["returns"]) <= 5e-3


def test_rollout_bitwise_reproducible(torch_cuda):
    """No float atomics, fixed-order reductions: two calls give identical bits."""
    import paper_2606_19729_b200 as vl
    for prec in (synth.PREC_FP32, synth.PREC_BF16):
        cfg = synth.CONFIGS[2]
        model = synth.make_model(cfg, prec=prec)
        inp = synth.make_inputs(cfg, P=300, Q=9, H=5)
        a = _run_gpu(torch_cuda, model, inp, prec, vl.KERNEL_AUTO, want_final=False)
        b = _run_gpu(torch_cuda, model, inp, prec, vl.KERNEL_AUTO, want_final=False)
        assert np.array_equal(a["values"], b["values"]) and np.array_equal(a["returns"], b["returns"])
        c = _run_gpu(torch_cuda, model, inp, prec, vl.KERNEL_AUTO, seed=4321, want_final=False)
        assert not np.array_equal(a["values"], c["values"])


def test_rollout_host_entry_matches_device(torch_cuda):
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[1]
    model = synth.make_model(cfg)
    inp = synth.make_inputs(cfg)
    dev = _run_gpu(torch, model, inp, synth.PREC_FP32, vl.KERNEL_AUTO, want_final=False)
    ctx = vl.Voila(model)
    parts = torch.from_numpy(inp.particles).pin_memory()
    seqs = torch.from_numpy(inp.action_seqs).pin_memory()
    vals = torch.empty(cfg.Q, dtype=torch.float32).pin_memory()
    wit = torch.empty((cfg.Q, cfg.O), dtype=torch.float32).pin_memory()
    ctx.voila_rollout_values_host(parts, seqs, None, 1234, vals, wit)
    assert np.array_equal(vals.numpy(), dev["values"])
    assert np.array_equal(wit.numpy(), dev["witness"])
    ctx.close()


def test_rollout_argument_errors(torch_cuda):
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[1]
    ctx = vl.Voila(synth.make_model(cfg))
    parts = torch.zeros((8, cfg.S), device="cuda")
    seqs = torch.zeros((2, 3), dtype=torch.int32, device="cuda")
    vals = torch.zeros(2, device="cuda")
    import ctypes as C
    lib = ctx.lib
    # workspace not reserved
    rc = lib.voila_rollout_values(ctx._h, C.c_void_p(parts.data_ptr()), 8, C.c_void_p(seqs.data_ptr()),
                                  2, 3, None, 1, C.c_void_p(vals.data_ptr()), None, None, None, None)
    assert rc == 4
    ctx.voila_reserve(8, 2, 3, 0)
    rc = lib.voila_rollout_values(ctx._h, None, 8, C.c_void_p(seqs.data_ptr()), 2, 3, None, 1,
                                  C.c_void_p(vals.data_ptr()), None, None, None, None)
    assert rc == 1
    rc = lib.voila_rollout_values(ctx._h, C.c_void_p(parts.data_ptr() + 4), 8,
                                  C.c_void_p(seqs.data_ptr()), 2, 3, None, 1,
                                  C.c_void_p(vals.data_ptr()), None, None, None, None)
    assert rc == 1  # misaligned
    ctx.close()


def test_best_action_matches_argmax(torch_cuda):
    """voila_best_action: q* = argmax_q V_q with ties to the lowest q and NaN never winning; the
    returned action is action_seqs[q*][0] (root action selection, include/voila.h)."""
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    ctx = vl.Voila(synth.make_model(synth.CONFIGS[1]))
    rng = np.random.default_rng(11)
    for Q, H in [(1, 1), (7, 3), (1000, 10), (4096, 30), (100_003, 2)]:
        v = rng.standard_normal(Q).astype(np.float32)
        seqs = rng.integers(0, 4, size=(Q, H), dtype=np.int32)
        if Q > 6:
            v[[3, 5]] = v.max() + 1.0          # a tie: the lower index must win
            v[1] = np.nan                      # NaN never wins
        bq, ba = ctx.voila_best_action(torch.from_numpy(v).cuda(), torch.from_numpy(seqs).cuda())
        ref = int(np.nanargmax(v))
        assert int(bq.item()) == ref and int(ba.item()) == int(seqs[ref, 0])
    ctx.close()
