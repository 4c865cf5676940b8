"""ctypes front-end of the CPU oracle (oracle/voila_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It never imports the CUDA package and
shares no code with it; models arrive as plain numpy arrays (duck-typed `ModelSpec`: attributes
S, O, A, Nz, f_T, f_Z, lik_obs, lik_state (each with dims/act/W/b), lik_action_cond, lam, gamma,
reward_kind, reward_param, action_cost).
"""
from __future__ import annotations

import ctypes as C
import importlib.util
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBS = {}


def _build():
    spec = importlib.util.spec_from_file_location("_voila_oracle_build",
                                                  os.path.join(_HERE, "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod.build()


def _lib(real: str = "f32"):
    if real in _LIBS:
        return _LIBS[real]
    paths = _build()
    lib = C.CDLL(paths[f"libvoila_oracle_{real}.so"])
    vp, i32, u32, u64, f32, f64 = C.c_void_p, C.c_int, C.c_uint32, C.c_uint64, C.c_float, C.c_double
    lib.vo_philox4x32_10.argtypes = [vp, vp, vp]
    lib.vo_philox4x32_10.restype = None
    lib.vo_normals.argtypes = [u64, u32, u32, u32, u32, i32, vp]
    lib.vo_normals.restype = None
    lib.vo_resample_word.argtypes = [u64]
    lib.vo_resample_word.restype = u32
    lib.vo_model_create.argtypes = [i32, i32, i32, i32, i32, f32, f32]
    lib.vo_model_create.restype = vp
    lib.vo_model_set_mlp.argtypes = [vp, i32, i32, vp, i32, vp, vp]
    lib.vo_model_set_mlp.restype = i32
    lib.vo_model_set_reward.argtypes = [vp, i32, vp, vp]
    lib.vo_model_set_reward.restype = i32
    lib.vo_model_set_emulate_bf16.argtypes = [vp, i32]
    lib.vo_model_set_emulate_bf16.restype = None
    lib.vo_model_destroy.argtypes = [vp]
    lib.vo_model_destroy.restype = None
    lib.vo_mlp_forward.argtypes = [vp, i32, vp, i32, vp]
    lib.vo_mlp_forward.restype = i32
    lib.vo_rollout_trajectory.argtypes = [vp, vp, vp, i32, u32, u32, u64, vp, vp]
    lib.vo_rollout_trajectory.restype = f64
    lib.vo_rollout_values.argtypes = [vp, vp, i32, vp, i32, i32, vp, u64, i32, vp, vp, vp]
    lib.vo_rollout_values.restype = i32
    lib.vo_rollout_values_term.argtypes = [vp, vp, i32, vp, i32, i32, vp, u64, i32, vp, vp, vp, vp, vp, vp]
    lib.vo_rollout_values_term.restype = i32
    lib.vo_pw_update.argtypes = [vp, vp, i32, vp, i32, vp, vp, vp, vp, i32, f64, f64, vp, u64,
                                 vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vo_pw_update.restype = i32
    lib.vo_diffusion_sample.argtypes = [vp, i32, vp, vp, i32, i32, u64, vp, i32, vp]
    lib.vo_diffusion_sample.restype = i32
    lib.vo_model_set_terminal.argtypes = [vp, i32, vp, vp, vp, vp, vp]
    lib.vo_model_set_terminal.restype = i32
    lib.vo_resample_systematic_x0.argtypes = [vp, i32, u32, vp]
    lib.vo_resample_systematic_x0.restype = i32
    lib.vo_resample_systematic.argtypes = [vp, i32, u64, vp]
    lib.vo_resample_systematic.restype = i32
    lib.vo_belief_update.argtypes = [vp, vp, i32, i32, vp, vp, u64, vp, vp, vp, vp, vp, vp, vp]
    lib.vo_belief_update.restype = i32
    lib.vo_belief_update_ess.argtypes = [vp, vp, i32, i32, vp, vp, u64, C.c_float, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vo_belief_update_ess.restype = i32
    lib.vo_effective_sample_size.argtypes = [vp, i32]
    lib.vo_effective_sample_size.restype = C.c_double
    lib.vo_normalised_weights.argtypes = [vp, i32, vp]
    lib.vo_normalised_weights.restype = i32
    lib.vo_num_threads.restype = i32
    lib.vo_set_num_threads.argtypes = [i32]
    lib.vo_real_bytes.restype = i32
    _LIBS[real] = lib
    return lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    _lib().vo_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def normals(seed, p, q, t, stream, n):
    out = np.zeros(n + 4, dtype=np.float32)
    _lib().vo_normals(int(seed), int(p), int(q), int(t), int(stream), int(n), _p(out))
    return out[:n]


def resample_word(seed):
    return int(_lib().vo_resample_word(int(seed)))


def resample_systematic_x0(v, x0):
    v = _f32(v)
    anc = np.zeros(v.shape[0], dtype=np.int32)
    st = _lib().vo_resample_systematic_x0(_p(v), v.shape[0], int(x0), _p(anc))
    return anc, st


def resample_systematic(v, seed):
    v = _f32(v)
    anc = np.zeros(v.shape[0], dtype=np.int32)
    st = _lib().vo_resample_systematic(_p(v), v.shape[0], int(seed), _p(anc))
    return anc, st


def effective_sample_size(v):
    v = _f32(v)
    return float(_lib().vo_effective_sample_size(_p(v), v.shape[0]))


def normalised_weights(v):
    v = _f32(v)
    w = np.zeros(v.shape[0], dtype=np.float64)
    st = _lib().vo_normalised_weights(_p(v), v.shape[0], _p(w))
    return w, st


def num_threads():
    return int(_lib().vo_num_threads())


def set_num_threads(n):
    for real in list(_LIBS) or ["f32"]:
        _lib(real).vo_set_num_threads(int(n))


class OracleModel:
    """Owns a vo_model.  real = 'f32' (the oracle proper) or 'f64' (tolerance derivation)."""

    def __init__(self, model, real: str = "f32", emulate_bf16: bool = False):
        self.lib = _lib(real)
        self.real = real
        self.S, self.O, self.A, self.Nz = model.S, model.O, model.A, model.Nz
        self.h = self.lib.vo_model_create(model.S, model.O, model.A, model.Nz,
                                          int(model.lik_action_cond), float(model.lam),
                                          float(model.gamma))
        self.out_dims = []
        for which, f in enumerate([model.f_T, model.f_Z, model.lik_obs, model.lik_state]):
            dims = np.asarray(f.dims, dtype=np.int32)
            Wf = np.concatenate([np.asarray(w, np.float32).ravel() for w in f.W])
            bf = np.concatenate([np.asarray(b, np.float32).ravel() for b in f.b])
            rc = self.lib.vo_model_set_mlp(self.h, which, len(f.W), _p(dims), int(f.act),
                                           _p(Wf), _p(bf))
            assert rc == 0
            self.out_dims.append((int(dims[0]), int(dims[-1])))
        for which, name in ((4, "denoise_T"), (5, "denoise_Z")):
            f = getattr(model, name, None)
            if f is not None:
                dims = np.asarray(f.dims, dtype=np.int32)
                Wf = np.concatenate([np.asarray(w, np.float32).ravel() for w in f.W])
                bf = np.concatenate([np.asarray(b, np.float32).ravel() for b in f.b])
                rc = self.lib.vo_model_set_mlp(self.h, which, len(f.W), _p(dims), int(f.act), _p(Wf), _p(bf))
                assert rc == 0
                while len(self.out_dims) <= which:
                    self.out_dims.append((0, 0))
                self.out_dims[which] = (int(dims[0]), int(dims[-1]))
        cost = _f32(model.action_cost)
        rc = self.lib.vo_model_set_reward(self.h, int(model.reward_kind),
                                          _p(_f32(model.reward_param).ravel()), _p(cost))
        assert rc == 0
        if emulate_bf16:
            self.lib.vo_model_set_emulate_bf16(self.h, 1)
        term = getattr(model, "terminal", None)
        if term is not None and len(term.radii):
            dims = np.asarray([len(c) for c in term.centers], dtype=np.int32)
            cen = np.concatenate([np.asarray(c, np.float32).ravel() for c in term.centers])
            rc = self.lib.vo_model_set_terminal(self.h, len(dims), _p(dims), _p(cen),
                                                _p(_f32(term.radii)), _p(_f32(term.rewards)),
                                                _p(np.asarray(term.stops, dtype=np.int32)))
            assert rc == 0

    def __del__(self):
        try:
            self.lib.vo_model_destroy(self.h)
        except Exception:
            pass

    def mlp_forward(self, which, x):
        x = _f32(x)
        rows = x.shape[0]
        assert x.shape[1] == self.out_dims[which][0]
        y = np.zeros((rows, self.out_dims[which][1]), dtype=np.float32)
        rc = self.lib.vo_mlp_forward(self.h, which, _p(x), rows, _p(y))
        assert rc == 0
        return y

    def rollout_trajectory(self, s0, actions, p, q, seed):
        s0 = _f32(s0)
        actions = np.ascontiguousarray(actions, dtype=np.int32)
        H = actions.shape[0]
        states = np.zeros((H + 1, self.S), dtype=np.float32)
        obs = np.zeros((H, self.O), dtype=np.float32)
        G = self.lib.vo_rollout_trajectory(self.h, _p(s0), _p(actions), H, int(p), int(q),
                                           int(seed), _p(states), _p(obs))
        return float(G), states, obs

    def rollout_values(self, particles, action_seqs, weights, seed, q_offset=0,
                       want_returns=False):
        particles = _f32(particles)
        action_seqs = np.ascontiguousarray(action_seqs, dtype=np.int32)
        weights = _f32(weights)
        P, (Q, H) = particles.shape[0], action_seqs.shape
        values = np.zeros(Q, dtype=np.float32)
        witness = np.zeros((Q, self.O), dtype=np.float32)
        returns = np.zeros((Q, P), dtype=np.float32) if want_returns else None
        rc = self.lib.vo_rollout_values(self.h, _p(particles), P, _p(action_seqs), Q, H,
                                        _p(weights), int(seed), int(q_offset), _p(values),
                                        _p(witness), _p(returns))
        if rc != 0:
            raise RuntimeError(f"vo_rollout_values -> {rc}")
        if want_returns:
            return values, witness, returns
        return values, witness

    def rollout_values_term(self, particles, action_seqs, weights, seed, q_offset=0):
        """Rollout with the per-trajectory detail of the termination tests: dict with values [Q],
        witness [Q][O], returns [Q][P], final_states [Q][P][S], t_term [Q][P] (H = never),
        margin [Q][P] (closest any membership decision came to its boundary)."""
        particles = _f32(particles)
        action_seqs = np.ascontiguousarray(action_seqs, dtype=np.int32)
        weights = _f32(weights)
        P, (Q, H) = particles.shape[0], action_seqs.shape
        out = {"values": np.zeros(Q, np.float32), "witness": np.zeros((Q, self.O), np.float32),
               "returns": np.zeros((Q, P), np.float32), "final_states": np.zeros((Q, P, self.S), np.float32),
               "t_term": np.zeros((Q, P), np.int32), "margin": np.zeros((Q, P), np.float32)}
        rc = self.lib.vo_rollout_values_term(self.h, _p(particles), P, _p(action_seqs), Q, H, _p(weights),
                                             int(seed), int(q_offset), _p(out["values"]), _p(out["witness"]),
                                             _p(out["returns"]), _p(out["final_states"]), _p(out["t_term"]),
                                             _p(out["margin"]))
        if rc != 0:
            raise RuntimeError(f"vo_rollout_values_term -> {rc}")
        return out

    def diffusion_sample(self, which, cond, actions, K, seed, traj_row=None):
        """The diffusion teacher's DDIM-ODE sampler (vo_diffusion_sample).  -> samples [N][D]
        (and the path [K+1][D] of sample traj_row when given)."""
        cond = _f32(cond)
        actions = np.ascontiguousarray(actions, dtype=np.int32)
        N = cond.shape[0]
        D = self.S if which == 0 else self.O
        out = np.zeros((N, D), np.float32)
        traj = np.zeros((K + 1, D), np.float32) if traj_row is not None else None
        rc = self.lib.vo_diffusion_sample(self.h, int(which), _p(cond), _p(actions), N, int(K), int(seed), _p(out),
                                          -1 if traj_row is None else int(traj_row), _p(traj))
        if rc != 0:
            raise RuntimeError(f"vo_diffusion_sample -> {rc}")
        return out if traj is None else (out, traj)

    def pw_update(self, particles, group_off, group_action, visit_count, branch_count, branch_obs, k_o,
                  alpha_o, weights, seed):
        """Vectorised progressive widening with batched likelihood (vo_pw_update).  visit_count,
        branch_count, branch_obs ([G][M_max][O]) are NOT modified: updated copies come back in the
        result dict next to the per-simulation outputs."""
        particles = _f32(particles)
        weights = _f32(weights)
        group_off = np.ascontiguousarray(group_off, dtype=np.int32)
        group_action = np.ascontiguousarray(group_action, dtype=np.int32)
        vc = np.array(visit_count, dtype=np.int32)
        bc = np.array(branch_count, dtype=np.int32)
        bo = np.array(branch_obs, dtype=np.float32)
        N, G, M_max = particles.shape[0], group_action.shape[0], bo.shape[1]
        out = {"proposals": np.zeros((N, self.S), np.float32), "obs": np.zeros((N, self.O), np.float32),
               "sim_branch": np.zeros(N, np.int32), "opened": np.zeros(N, np.int32),
               "logits": np.zeros(N, np.float32), "post_weights": np.zeros(N, np.float32),
               "ancestors": np.zeros(N, np.int32), "particles": np.zeros((N, self.S), np.float32),
               "weights": np.zeros(N, np.float32), "seg_status": np.zeros(G * M_max, np.int32)}
        rc = self.lib.vo_pw_update(self.h, _p(particles), N, _p(group_off), G, _p(group_action), _p(vc), _p(bc),
                                   _p(bo), M_max, float(k_o), float(alpha_o), _p(weights), int(seed),
                                   _p(out["proposals"]), _p(out["obs"]), _p(out["sim_branch"]), _p(out["opened"]),
                                   _p(out["logits"]), _p(out["post_weights"]), _p(out["ancestors"]),
                                   _p(out["particles"]), _p(out["weights"]), _p(out["seg_status"]))
        if rc != 0:
            raise RuntimeError(f"vo_pw_update -> {rc}")
        out.update({"visit_count": vc, "branch_count": bc, "branch_obs": bo})
        return out

    def belief_update(self, particles, action, observation, weights, seed, ess_threshold=None):
        """ess_threshold=None: the plain SIR update (always resample); a float: adaptive resampling
        (resample iff ESS < ess_threshold * N), outputs "ess" and "resampled" added."""
        particles = _f32(particles)
        observation = _f32(observation)
        weights = _f32(weights)
        N = particles.shape[0]
        out = {
            "proposals": np.zeros((N, self.S), dtype=np.float32),
            "logits": np.zeros(N, dtype=np.float32),
            "post_weights": np.zeros(N, dtype=np.float32),
            "ancestors": np.zeros(N, dtype=np.int32),
            "particles": np.zeros((N, self.S), dtype=np.float32),
            "weights": np.zeros(N, dtype=np.float32),
        }
        le = np.zeros(1, dtype=np.float64)
        if ess_threshold is None:
            rc = self.lib.vo_belief_update(self.h, _p(particles), N, int(action), _p(observation),
                                           _p(weights), int(seed), _p(out["proposals"]),
                                           _p(out["logits"]), _p(out["post_weights"]), _p(le),
                                           _p(out["ancestors"]), _p(out["particles"]),
                                           _p(out["weights"]))
        else:
            ess = np.zeros(1, dtype=np.float64)
            res = np.zeros(1, dtype=np.int32)
            rc = self.lib.vo_belief_update_ess(self.h, _p(particles), N, int(action), _p(observation),
                                               _p(weights), int(seed), C.c_float(ess_threshold),
                                               _p(out["proposals"]), _p(out["logits"]),
                                               _p(out["post_weights"]), _p(le), _p(out["ancestors"]),
                                               _p(out["particles"]), _p(out["weights"]), _p(ess), _p(res))
            out["ess"] = float(ess[0])
            out["resampled"] = int(res[0])
        out["log_evidence"] = float(le[0])
        out["status"] = rc
        return out
