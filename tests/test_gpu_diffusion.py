"""GPU parity: voila_diffusion_sample (the diffusion teacher's DDIM-ODE sampler, SURVEY 8f f4;
PAPER.md:101-109) through the C ABI against the oracle, sample by sample."""
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


def _case(torch, oracle, cfg_idx, prec, hidden, N, K, seed, kernel=None):
    import paper_2606_19729_b200 as vl
    cfg = synth.CONFIGS[cfg_idx]
    vT, vZ = synth.make_denoisers(cfg, hidden)
    model = synth.make_model(cfg, prec=prec).replace(denoise_T=vT, denoise_Z=vZ)
    rng = np.random.default_rng(seed)
    cond = rng.standard_normal((N, cfg.S)).astype(np.float32)
    act = rng.integers(0, cfg.A, N).astype(np.int32)
    bf16 = prec == synth.PREC_BF16
    cond_np = synth.bf16_round_np(cond) if bf16 else cond
    ctx = vl.Voila(model, device=0, prec=prec)
    if kernel is not None:
        ctx.voila_set_kernel(kernel)
    om = oracle.OracleModel(model, emulate_bf16=bf16)
    names = []
    for which in (0, 1):
        l0 = ctx.voila_launch_count()
        out = ctx.voila_diffusion_sample(which, ctx.to_particles(cond), torch.from_numpy(act).cuda(), K, seed)
        torch.cuda.synchronize()
        assert ctx.voila_launch_count() - l0 >= K  # K denoiser calls per sample
        ref = om.diffusion_sample(which, cond_np, act, K, seed)
        assert_close(t2n(out), ref, TOL_BF16_STATE if bf16 else TOL_FP32, f"teacher {which}")
        names.append(ctx.voila_last_belief_kernel())
    ctx.close()
    return names


def test_diffusion_fp32(torch_cuda, oracle):
    _case(torch_cuda, oracle, 1, synth.PREC_FP32, [64, 64], N=333, K=8, seed=5)
    _case(torch_cuda, oracle, 1, synth.PREC_FP32, [32], N=40, K=1, seed=6)


def test_diffusion_bf16_cuda_cores(torch_cuda, oracle):
    import paper_2606_19729_b200 as vl
    _case(torch_cuda, oracle, 2, synth.PREC_BF16, [128, 128], N=500, K=12, seed=7, kernel=vl.KERNEL_FFMA)


@pytest.mark.parametrize("cfg_idx,hidden,N,K", [(2, [128, 128], 700, 12), (3, [512, 512, 512, 512], 1500, 16),
                                               (3, [256, 256, 256], 40000, 6)])
def test_diffusion_bf16(torch_cuda, oracle, cfg_idx, hidden, N, K):
    names = _case(torch_cuda, oracle, cfg_idx, synth.PREC_BF16, hidden, N=N, K=K, seed=8 + cfg_idx)
    # the tcgen05 denoiser program serves both teachers; the two-slot build once N > 256 x CTA pairs
    want = "belief_tc2_dual_kernel" if (N > 20000 and max(hidden) <= 256) else "belief_tc2_kernel"
    assert all(want in n for n in names), names


def test_diffusion_errors(torch_cuda):
    import paper_2606_19729_b200 as vl
    torch = torch_cuda
    cfg = synth.CONFIGS[1]
    ctx = vl.Voila(synth.make_model(cfg), device=0)  # no denoisers
    cond = ctx.to_particles(np.zeros((4, cfg.S), np.float32))
    act = torch.zeros(4, dtype=torch.int32, device="cuda")
    with pytest.raises(vl.VoilaError, match="unsupported"):
        ctx.voila_diffusion_sample(0, cond, act, 4, 1)
    ctx.close()
    vT, vZ = synth.make_denoisers(cfg, [16])
    ctx = vl.Voila(synth.make_model(cfg).replace(denoise_T=vT, denoise_Z=vZ), device=0)
    with pytest.raises(vl.VoilaError, match="invalid"):
        ctx.voila_diffusion_sample(0, cond, act, 0, 1)
    with pytest.raises(vl.VoilaError, match="invalid"):
        ctx.voila_diffusion_sample(2, cond, act, 4, 1)
    ctx.close()
