"""Pins for the oracle's MLP forward (O3).  CPU only."""
import numpy as np
import torch

from paper_2606_19729_b200 import synth


def _torch_mlp(f, x, dtype=torch.float64):
    h = torch.tensor(x, dtype=dtype)
    for l in range(f.n_layers):
        h = torch.nn.functional.linear(h, torch.tensor(f.W[l], dtype=dtype),
                                       torch.tensor(f.b[l], dtype=dtype))
        if l < f.n_layers - 1:
            if f.act == synth.ACT_RELU:
                h = torch.relu(h)
            elif f.act == synth.ACT_SILU:
                h = torch.nn.functional.silu(h)
    return h.numpy()


def test_mlp_matches_torch_linear_chain(oracle):
    for idx in (1, 2, 3):
        cfg = synth.CONFIGS[idx]
        model = synth.make_model(cfg)
        om = oracle.OracleModel(model)
        rng = np.random.default_rng(idx)
        for which, f in enumerate(model.mlps()):
            x = rng.standard_normal((37, f.dims[0])).astype(np.float32)
            ref = _torch_mlp(f, x)
            got = om.mlp_forward(which, x)
            assert got.shape == ref.shape
            np.testing.assert_allclose(got, ref, rtol=2e-5, atol=2e-6)


def test_mlp_hand_2x2(oracle):
    # y = W2 relu(W1 x + b1) + b2 worked by hand
    W1 = np.array([[1.0, -2.0], [0.5, 3.0]], np.float32)
    b1 = np.array([0.25, -1.0], np.float32)
    W2 = np.array([[2.0, -1.0], [0.0, 4.0]], np.float32)
    b2 = np.array([1.0, -3.0], np.float32)
    f = synth.MLPSpec([2, 2, 2], synth.ACT_RELU, [W1, W2], [b1, b2])
    cfg = synth.CONFIGS[1]
    model = synth.make_model(cfg).replace(lik_obs=f)
    om = oracle.OracleModel(model)
    # x = (1, 1): pre = (1-2+.25, .5+3-1) = (-0.75, 2.5) -> relu (0, 2.5) -> (0-2.5+1, 10-3) = (-1.5, 7)
    # x = (2,-1): pre = (2+2+.25, 1-3-1) = (4.25, -3) -> (4.25, 0) -> (8.5+1, -3) = (9.5, -3)
    y = om.mlp_forward(2, np.array([[1, 1], [2, -1]], np.float32))
    np.testing.assert_allclose(y, [[-1.5, 7.0], [9.5, -3.0]], rtol=0, atol=1e-6)


def test_mlp_activation_none_is_affine(oracle):
    cfg = synth.CONFIGS[1]
    rng = np.random.default_rng(3)
    f = synth.make_mlp(rng, [2, 5, 3], synth.ACT_NONE)
    model = synth.make_model(cfg).replace(lik_obs=f)
    om = oracle.OracleModel(model)
    x = rng.standard_normal((9, 2)).astype(np.float32)
    Wt = f.W[1].astype(np.float64) @ f.W[0].astype(np.float64)
    bt = f.W[1].astype(np.float64) @ f.b[0] + f.b[1]
    np.testing.assert_allclose(om.mlp_forward(2, x), x @ Wt.T + bt, rtol=1e-5, atol=1e-6)


def test_bf16_hook_rounds_only_operands(oracle):
    cfg = synth.CONFIGS[2]
    model = synth.make_model(cfg)
    om_e = oracle.OracleModel(model, emulate_bf16=True)
    rng = np.random.default_rng(5)
    x = rng.standard_normal((16, model.f_T.dims[0])).astype(np.float32)
    # reference: same chain in fp64 with weights and every layer input rounded to bf16
    f = model.f_T
    h = x.astype(np.float64)
    for l in range(f.n_layers):
        hb = synth.bf16_round_np(h.astype(np.float32)).astype(np.float64)
        h = hb @ synth.bf16_round_np(f.W[l]).astype(np.float64).T + f.b[l]
        if l < f.n_layers - 1:
            h = h / (1 + np.exp(-h))
    np.testing.assert_allclose(om_e.mlp_forward(0, x), h, rtol=3e-3, atol=3e-4)
