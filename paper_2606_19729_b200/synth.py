"""Seeded synthetic inputs for the VOiLA hot path: model weights, particles, action sequences,
observations and prior weights, shaped like BASELINE.json's five configs.

This module holds DATA GENERATION ONLY (numpy random draws and shape bookkeeping).  None of the
method's arithmetic (no MLP evaluation, no Philox, no resampling) lives here, so it may serve
both the CUDA path and the CPU oracle: each side receives the same plain numpy arrays.

The paper's own domains (FloorPositioning, LeggedNavigation, TargetFinding)
need its datasets, simulator and trained weights, none of which exist here; these configs stand
in for them, taking their shapes.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

ACT_NONE, ACT_RELU, ACT_SILU = 0, 1, 2
R_NEG_L2_GOAL, R_NEG_QUADRATIC, R_LINEAR = 0, 1, 2
PREC_FP32, PREC_BF16 = 0, 1

BASE_SEED = 20260619


@dataclass
class MLPSpec:
    """y = W_L(...act(W_1 x + b_1)...) + b_L ; W[l] is [out][in] row-major fp32."""
    dims: List[int]
    act: int
    W: List[np.ndarray]
    b: List[np.ndarray]

    @property
    def n_layers(self) -> int:
        return len(self.W)

    def flat(self):
        return (np.concatenate([w.ravel() for w in self.W]).astype(np.float32),
                np.concatenate([b.ravel() for b in self.b]).astype(np.float32))


@dataclass
class TerminalSpec:
    """Terminal regions (R25): ball k over the leading len(centers[k]) state coordinates,
    radius radii[k]; pays rewards[k] when an alive state is inside; stops[k] = 1 ends the episode."""
    centers: List[np.ndarray]
    radii: np.ndarray
    rewards: np.ndarray
    stops: np.ndarray


@dataclass
class ModelSpec:
    S: int
    O: int
    A: int
    Nz: int
    f_T: MLPSpec
    f_Z: MLPSpec
    lik_obs: MLPSpec      # f : O -> ... -> d
    lik_state: MLPSpec    # g : S (+A) -> ... -> d
    lik_action_cond: int = 0
    lam: float = 1.0
    gamma: float = 0.95
    reward_kind: int = R_NEG_L2_GOAL
    reward_param: np.ndarray = None
    action_cost: Optional[np.ndarray] = None
    prec: int = PREC_FP32
    terminal: Optional[TerminalSpec] = None
    # diffusion teachers: denoisers v(c, a, x_tau, tau), input [c ; onehot(a) ; x ; temb(8)]
    denoise_T: Optional[MLPSpec] = None   # -> S
    denoise_Z: Optional[MLPSpec] = None   # -> O

    def mlps(self):
        return [self.f_T, self.f_Z, self.lik_obs, self.lik_state]

    def replace(self, **kw) -> "ModelSpec":
        return dataclasses.replace(self, **kw)


@dataclass
class Config:
    name: str
    index: int            # 1-based index into BASELINE.json configs
    S: int
    O: int
    A: int
    Nz: int
    hidden: List[int]
    act: int
    tower_hidden: List[int]
    tower_d: int
    P: int
    Q: int
    H: int
    N: int                # particles in the belief update
    gamma: float
    reward_kind: int
    prec: int
    particle_var: float = 1.0
    prior_logw_var: float = 0.0   # >0: prior weights exp(N(0, var)); 0: uniform (NULL)
    plan_steps: int = 1
    bu_action: int = 1
    extra: dict = field(default_factory=dict)


CONFIGS = {
    1: Config("cfg1_tiny_fp32", 1, S=2, O=2, A=4, Nz=2, hidden=[64, 64], act=ACT_RELU,
              tower_hidden=[64], tower_d=32, P=256, Q=64, H=10, N=256, gamma=0.95,
              reward_kind=R_NEG_L2_GOAL, prec=PREC_FP32),
    2: Config("cfg2_mid", 2, S=8, O=8, A=8, Nz=8, hidden=[128, 128, 128], act=ACT_SILU,
              tower_hidden=[128], tower_d=64, P=1024, Q=512, H=15, N=1024, gamma=0.95,
              reward_kind=R_NEG_L2_GOAL, prec=PREC_BF16, particle_var=0.5),
    3: Config("cfg3_quadruped_bf16", 3, S=48, O=64, A=16, Nz=16, hidden=[256, 256, 256],
              act=ACT_SILU, tower_hidden=[256], tower_d=128, P=2048, Q=1024, H=20, N=2048,
              gamma=0.95, reward_kind=R_NEG_QUADRATIC, prec=PREC_BF16),
    4: Config("cfg4_belief_stress_bf16", 4, S=48, O=64, A=16, Nz=16, hidden=[256, 256, 256],
              act=ACT_SILU, tower_hidden=[256], tower_d=128, P=2048, Q=16, H=4, N=1 << 20,
              gamma=0.95, reward_kind=R_NEG_QUADRATIC, prec=PREC_BF16, prior_logw_var=4.0),
    5: Config("cfg5_large_sweep_bf16", 5, S=64, O=64, A=32, Nz=32, hidden=[512, 512, 512, 512],
              act=ACT_SILU, tower_hidden=[256], tower_d=128, P=4096, Q=4096, H=30, N=4096,
              gamma=0.95, reward_kind=R_NEG_QUADRATIC, prec=PREC_BF16, plan_steps=10),
}


def _xavier(rng: np.random.Generator, fan_out: int, fan_in: int, gain: float = 1.0) -> np.ndarray:
    a = gain * np.sqrt(6.0 / (fan_in + fan_out))
    return rng.uniform(-a, a, size=(fan_out, fan_in)).astype(np.float32)


def make_mlp(rng: np.random.Generator, dims: List[int], act: int, gain: float = 1.0,
             bias_range: float = 0.1) -> MLPSpec:
    W, b = [], []
    for l in range(len(dims) - 1):
        W.append(_xavier(rng, dims[l + 1], dims[l], gain))
        b.append(rng.uniform(-bias_range, bias_range, size=(dims[l + 1],)).astype(np.float32))
    return MLPSpec(list(dims), act, W, b)


TEMB = 8  # width of the diffusion-time embedding (R31)


def make_denoisers(cfg: Config, hidden: List[int], seed: Optional[int] = None, gain: float = 1.0):
    """Random-init denoisers of the two diffusion teachers (transition: -> S, observation: -> O)."""
    seed = BASE_SEED + 500 + cfg.index if seed is None else seed
    r = [np.random.default_rng(s) for s in np.random.SeedSequence(seed).spawn(2)]
    vT = make_mlp(r[0], [cfg.S + cfg.A + cfg.S + TEMB] + list(hidden) + [cfg.S], cfg.act, gain)
    vZ = make_mlp(r[1], [cfg.S + cfg.A + cfg.O + TEMB] + list(hidden) + [cfg.O], cfg.act, gain)
    return vT, vZ


def make_model(cfg: Config, seed: Optional[int] = None, gain: float = 1.0,
               prec: Optional[int] = None, lik_action_cond: int = 0, lam: float = 1.0,
               action_cost: bool = False) -> ModelSpec:
    """Random-init generators and towers of the config's architecture (Xavier-uniform weights,
    biases U[-0.1, 0.1]); reward parameters: goal ~ U[-1,1]^S or M = B B^T / S with B ~ N(0,1)."""
    seed = BASE_SEED + cfg.index if seed is None else seed
    ss = np.random.SeedSequence(seed).spawn(8)
    r = [np.random.default_rng(s) for s in ss]
    gin = cfg.S + cfg.A + cfg.Nz
    f_T = make_mlp(r[0], [gin] + cfg.hidden + [cfg.S], cfg.act, gain)
    f_Z = make_mlp(r[1], [gin] + cfg.hidden + [cfg.O], cfg.act, gain)
    lik_obs = make_mlp(r[2], [cfg.O] + cfg.tower_hidden + [cfg.tower_d], cfg.act, gain)
    g_in = cfg.S + (cfg.A if lik_action_cond else 0)
    lik_state = make_mlp(r[3], [g_in] + cfg.tower_hidden + [cfg.tower_d], cfg.act, gain)
    if cfg.reward_kind == R_NEG_L2_GOAL:
        param = r[4].uniform(-1.0, 1.0, size=(cfg.S,)).astype(np.float32)
    elif cfg.reward_kind == R_NEG_QUADRATIC:
        B = r[4].standard_normal((cfg.S, cfg.S))
        param = (B @ B.T / cfg.S).astype(np.float32)
    else:
        param = r[4].uniform(-1.0, 1.0, size=(cfg.S + 1,)).astype(np.float32)
    cost = r[5].uniform(-0.2, 0.0, size=(cfg.A,)).astype(np.float32) if action_cost else None
    return ModelSpec(cfg.S, cfg.O, cfg.A, cfg.Nz, f_T, f_Z, lik_obs, lik_state,
                     lik_action_cond=lik_action_cond, lam=lam, gamma=cfg.gamma,
                     reward_kind=cfg.reward_kind, reward_param=param, action_cost=cost,
                     prec=cfg.prec if prec is None else prec)


@dataclass
class Inputs:
    particles: np.ndarray          # [P][S] fp32
    action_seqs: np.ndarray        # [Q][H] int32
    weights: Optional[np.ndarray]  # [P] fp32 or None (uniform)
    bu_particles: np.ndarray       # [N][S] fp32
    bu_weights: Optional[np.ndarray]
    observation: np.ndarray        # [O] fp32
    bu_action: int
    seed: int


def make_inputs(cfg: Config, seed: Optional[int] = None, P: Optional[int] = None,
                Q: Optional[int] = None, H: Optional[int] = None,
                N: Optional[int] = None) -> Inputs:
    seed = BASE_SEED + 1000 + cfg.index if seed is None else seed
    P = cfg.P if P is None else P
    Q = cfg.Q if Q is None else Q
    H = cfg.H if H is None else H
    N = cfg.N if N is None else N
    ss = np.random.SeedSequence(seed).spawn(6)
    r = [np.random.default_rng(s) for s in ss]
    sd = np.sqrt(cfg.particle_var)
    particles = (sd * r[0].standard_normal((P, cfg.S))).astype(np.float32)
    action_seqs = r[1].integers(0, cfg.A, size=(Q, H), dtype=np.int32)
    if N == P:
        bu_particles = particles
    else:
        bu_particles = (sd * r[2].standard_normal((N, cfg.S))).astype(np.float32)
    bu_weights = None
    if cfg.prior_logw_var > 0:
        g = np.sqrt(cfg.prior_logw_var) * r[3].standard_normal(N)
        bu_weights = np.exp(g).astype(np.float32)
    observation = r[4].standard_normal(cfg.O).astype(np.float32)
    return Inputs(particles, action_seqs, None, bu_particles, bu_weights, observation,
                  cfg.bu_action, seed)


def observations_for_steps(cfg: Config, n_steps: int, seed: Optional[int] = None) -> np.ndarray:
    """Pre-seeded observations o_k ~ N(0, I) for the multi-step planning loop (config 5)."""
    seed = BASE_SEED + 2000 + cfg.index if seed is None else seed
    return np.random.default_rng(seed).standard_normal((n_steps, cfg.O)).astype(np.float32)


def bf16_round_np(x: np.ndarray) -> np.ndarray:
    """Round fp32 to the nearest bf16 (ties to even), returned as fp32.  Pure data conversion,
    used so that both sides start from identical bf16-representable particle states."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(x.shape)


def to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit patterns (uint16), round to nearest even."""
    return (bf16_round_np(x).view(np.uint32) >> 16).astype(np.uint16)


def from_bf16_bits(u: np.ndarray) -> np.ndarray:
    return (u.astype(np.uint32) << 16).view(np.float32)


def flops_per_rollout_step(model: ModelSpec, algorithmic: bool = True) -> int:
    """2*MAC of one f_T plus one f_Z evaluation; `algorithmic` folds the one-hot action block
    into the first-layer bias (first-layer K = S + Nz)."""
    tot = 0
    for f in (model.f_T, model.f_Z):
        for l in range(f.n_layers):
            k = f.dims[l]
            if l == 0 and algorithmic:
                k -= model.A
            tot += 2 * k * f.dims[l + 1]
    return tot


def flops_per_belief_particle(model: ModelSpec, algorithmic: bool = True) -> int:
    """2*MAC of one proposal f_T plus one state-tower g evaluation and the score dot product
    (SURVEY 8a R7-R8); `algorithmic` folds one-hot action blocks into first-layer biases."""
    tot = 0
    towers = [(model.f_T, True), (model.lik_state, bool(model.lik_action_cond))]
    for f, has_onehot in towers:
        for l in range(f.n_layers):
            k = f.dims[l]
            if l == 0 and algorithmic and has_onehot:
                k -= model.A
            tot += 2 * k * f.dims[l + 1]
    return tot + 2 * model.lik_state.dims[-1]
