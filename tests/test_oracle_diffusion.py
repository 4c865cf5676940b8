"""Pins for the oracle of the diffusion teacher's sampler (vo_diffusion_sample; PAPER.md:101-109;
SURVEY 8f f4; readings R30-R32).  CPU only.  Expected values: closed forms of the DDIM-ODE
recursion for denoisers that are linear in x or independent of x, the separately pinned MLP forward
and normals for K = 1."""
import numpy as np

from paper_2606_19729_b200 import synth
from paper_2606_19729_b200.synth import ACT_NONE, ACT_SILU, MLPSpec, TEMB


def _model(cfg, vT=None, vZ=None):
    return synth.make_model(cfg).replace(denoise_T=vT, denoise_Z=vZ)


def _temb(tau):
    return np.array([f(np.pi * 2 ** k * tau) for k in range(TEMB // 2) for f in (np.sin, np.cos)])


def test_one_step_is_minus_the_denoiser_at_tau_one(oracle):
    """K = 1: alpha(1) = 0, sigma(1) = 1, alpha(0) = 1, sigma(0) = 0, so x_0 = -v(c, a, omega, 1)."""
    cfg = synth.CONFIGS[1]
    rng = np.random.default_rng(0)
    vT, vZ = synth.make_denoisers(cfg, [32, 32])
    om = oracle.OracleModel(_model(cfg, vT, vZ))
    N = 9
    cond = rng.standard_normal((N, cfg.S)).astype(np.float32)
    act = rng.integers(0, cfg.A, N).astype(np.int32)
    for which, D in ((0, cfg.S), (1, cfg.O)):
        out = om.diffusion_sample(which, cond, act, K=1, seed=31)
        for i in range(N):
            omega = oracle.normals(31, i, 0, 0, 7, D)
            x = np.concatenate([cond[i], np.eye(cfg.A, dtype=np.float32)[act[i]], omega, _temb(1.0).astype(np.float32)])
            np.testing.assert_allclose(out[i], -om.mlp_forward(4 + which, x[None])[0], rtol=1e-5, atol=1e-6)


def _linear_denoiser(cfg, D, M=None, Ws=None, Wa=None, Wt=None, b=None):
    gin = cfg.S + cfg.A + D + TEMB
    W = np.zeros((D, gin), np.float32)
    if Ws is not None: W[:, :cfg.S] = Ws
    if Wa is not None: W[:, cfg.S:cfg.S + cfg.A] = Wa
    if M is not None: W[:, cfg.S + cfg.A:cfg.S + cfg.A + D] = M
    if Wt is not None: W[:, cfg.S + cfg.A + D:] = Wt
    return MLPSpec([gin, D], ACT_NONE, [W], [np.zeros(D, np.float32) if b is None else b.astype(np.float32)])


def test_denoiser_linear_in_x_gives_a_matrix_power(oracle):
    """v = M x: every DDIM step is x <- (cos(phi - phi') I - sin(phi - phi') M) x with phi - phi' = pi / (2K)
    (the v-prediction step written out is a rotation of (x, v)), so x_0 = (c I - s M)^K omega."""
    cfg = synth.CONFIGS[1]
    rng = np.random.default_rng(1)
    D = cfg.S
    M = (0.6 * rng.standard_normal((D, D))).astype(np.float32)
    om = oracle.OracleModel(_model(cfg, _linear_denoiser(cfg, D, M=M)))
    cond = rng.standard_normal((5, cfg.S)).astype(np.float32)
    act = np.zeros(5, np.int32)
    for K in (1, 3, 16):
        out, traj = om.diffusion_sample(0, cond, act, K=K, seed=4, traj_row=2)
        c, s = np.cos(np.pi / (2 * K)), np.sin(np.pi / (2 * K))
        step = c * np.eye(D) - s * M.astype(np.float64)
        for i in range(5):
            omega = oracle.normals(4, i, 0, 0, 7, D).astype(np.float64)
            np.testing.assert_allclose(out[i], np.linalg.matrix_power(step, K) @ omega, rtol=2e-5, atol=2e-6)
        assert np.array_equal(traj[0], oracle.normals(4, 2, 0, 0, 7, D)) and np.array_equal(traj[K], out[2])


def test_denoiser_independent_of_x_gives_a_geometric_sum(oracle):
    """v_k = Ws c + Wa e_a + Wt temb(tau_k) + b: x_0 = c^K omega - s sum_k c^(K-1-k) v_k; zero denoiser: c^K omega."""
    cfg = synth.CONFIGS[1]
    rng = np.random.default_rng(2)
    D = cfg.O
    Ws, Wa = rng.standard_normal((D, cfg.S)), rng.standard_normal((D, cfg.A))
    Wt, b = rng.standard_normal((D, TEMB)), rng.standard_normal(D)
    om = oracle.OracleModel(_model(cfg, None, _linear_denoiser(cfg, D, Ws=Ws, Wa=Wa, Wt=Wt, b=b)))
    N, K = 6, 7
    cond = rng.standard_normal((N, cfg.S)).astype(np.float32)
    act = rng.integers(0, cfg.A, N).astype(np.int32)
    out = om.diffusion_sample(1, cond, act, K=K, seed=8)
    c, s = np.cos(np.pi / (2 * K)), np.sin(np.pi / (2 * K))
    for i in range(N):
        x = oracle.normals(8, i, 0, 0, 7, D).astype(np.float64)
        ref = c ** K * x
        for k in range(K):
            vk = (Ws.astype(np.float32) @ cond[i] + Wa.astype(np.float32)[:, act[i]]
                  + Wt.astype(np.float32).astype(np.float64) @ _temb(1 - k / K) + b.astype(np.float32))
            ref = ref - s * c ** (K - 1 - k) * vk
        np.testing.assert_allclose(out[i], ref, rtol=3e-5, atol=3e-5)
    zero = oracle.OracleModel(_model(cfg, None, _linear_denoiser(cfg, D)))
    out0 = zero.diffusion_sample(1, cond, act, K=K, seed=8)
    for i in range(N):
        np.testing.assert_allclose(out0[i], c ** K * oracle.normals(8, i, 0, 0, 7, D), rtol=1e-5)


def test_nonlinear_denoiser_against_a_numpy_recursion(oracle):
    """A SiLU denoiser: the recursion of PAPER.md:101-105 written independently in numpy fp64 around the
    (separately pinned) MLP forward."""
    cfg = synth.CONFIGS[2]
    rng = np.random.default_rng(3)
    vT, _ = synth.make_denoisers(cfg, [48, 48])
    om = oracle.OracleModel(_model(cfg, vT, None))
    N, K = 4, 10
    cond = rng.standard_normal((N, cfg.S)).astype(np.float32)
    act = rng.integers(0, cfg.A, N).astype(np.int32)
    out = om.diffusion_sample(0, cond, act, K=K, seed=12)
    for i in range(N):
        x = oracle.normals(12, i, 0, 0, 7, cfg.S).astype(np.float64)
        for k in range(K):
            tau, tau_n = 1 - k / K, 1 - (k + 1) / K
            inp = np.concatenate([cond[i], np.eye(cfg.A)[act[i]], x, _temb(tau)]).astype(np.float32)
            v = om.mlp_forward(4, inp[None])[0].astype(np.float64)
            abar, abar_n = np.cos(np.pi * tau / 2) ** 2, np.cos(np.pi * tau_n / 2) ** 2   # cosine schedule
            x0 = np.sqrt(abar) * x - np.sqrt(1 - abar) * v                                 # v-prediction
            eps = np.sqrt(1 - abar) * x + np.sqrt(abar) * v
            x = np.sqrt(abar_n) * x0 + np.sqrt(1 - abar_n) * eps                           # DDIM, eta = 0
        np.testing.assert_allclose(out[i], x, rtol=2e-4, atol=2e-5)
