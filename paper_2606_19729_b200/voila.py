"""Thin ctypes binding of libvoila (include/voila.h).  Argument marshalling only: every step of the
hot path runs in the CUDA kernels behind the C ABI.  torch is used for device memory and streams.

There is NO CPU fallback: if libvoila.so is missing it is built with nvcc; if that fails, or no
sm_100 device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

KERNEL_AUTO, KERNEL_FFMA, KERNEL_TCGEN05, KERNEL_TCGEN05_PAIR = 0, 1, 2, 3
PREC_FP32, PREC_BF16 = 0, 1

# every symbol include/voila.h declares (tests check that the library exports all of them)
EXPORTS = [
    "voila_create", "voila_destroy", "voila_workspace_bytes", "voila_reserve", "voila_set_kernel",
    "voila_tcgen05_supported", "voila_rollout_values", "voila_belief_update", "voila_belief_update_ess",
    "voila_resample_systematic", "voila_mlp_forward", "voila_best_action", "voila_porpp_backup_level",
    "voila_rollout_values_host",
    "voila_belief_update_host", "voila_launch_count", "voila_last_rollout_kernel", "voila_last_belief_kernel",
    "voila_status_string", "voila_last_cuda_error", "voila_version", "voila_set_profiling",
    "voila_profile_read", "voila_pw_workspace_bytes", "voila_pw_reserve", "voila_pw_update",
    "voila_porpp_backup", "voila_diffusion_sample", "voila_plan_host",
    "voila_resample_systematic_static", "voila_static_last_error",
]


class VoilaError(RuntimeError):
    pass


STATIC_MAX_N = 1 << 20  # VOILA_STATIC_MAX_N


def voila_resample_systematic_static(v, seed, ancestors_out, status_out=None, stream=None):
    """voila_resample_systematic_static (include/voila.h): the resampler that allocates nothing.  The
    caller passes the outputs too (ancestors_out [N] int32, status_out [1] int32 or None); scratch is
    the library's static device array, shared by every call: do not overlap calls on the GPU."""
    import torch
    lib = load_library()
    N = v.numel()
    assert v.dtype == torch.float32 and v.is_contiguous() and v.is_cuda
    assert ancestors_out.dtype == torch.int32 and ancestors_out.is_contiguous() and ancestors_out.numel() >= N
    assert status_out is None or (status_out.dtype == torch.int32 and status_out.numel() >= 1)
    st = torch.cuda.current_stream(v.device).cuda_stream if stream is None else stream
    with torch.cuda.device(v.device):
        rc = lib.voila_resample_systematic_static(_dptr(v), N, C.c_uint64(int(seed)), _dptr(ancestors_out),
                                                  _dptr(status_out) if status_out is not None else None,
                                                  C.c_void_p(st))
    if rc != 0:
        raise VoilaError(f"voila_resample_systematic_static: status {rc}: "
                         f"{lib.voila_static_last_error().decode()}")
    return ancestors_out


class _Mlp(C.Structure):
    _fields_ = [("n_layers", C.c_int), ("dims", C.POINTER(C.c_int)),
                ("W", C.POINTER(C.POINTER(C.c_float))), ("b", C.POINTER(C.POINTER(C.c_float))),
                ("act", C.c_int)]


class _Reward(C.Structure):
    _fields_ = [("kind", C.c_int), ("param", C.POINTER(C.c_float)),
                ("action_cost", C.POINTER(C.c_float))]


class _Terminal(C.Structure):
    _fields_ = [("n_regions", C.c_int), ("dims", C.POINTER(C.c_int)), ("centers", C.POINTER(C.c_float)),
                ("radii", C.POINTER(C.c_float)), ("rewards", C.POINTER(C.c_float)),
                ("stops", C.POINTER(C.c_int))]


class _PorppLevel(C.Structure):
    _fields_ = [("R", C.c_void_p), ("logpi0", C.c_void_p), ("child_off", C.c_void_p), ("child_idx", C.c_void_p),
                ("child_w", C.c_void_p), ("n_belief", C.c_int), ("psi_out", C.c_void_p), ("v_out", C.c_void_p)]


class _ModelDesc(C.Structure):
    _fields_ = [("state_dim", C.c_int), ("obs_dim", C.c_int), ("n_actions", C.c_int),
                ("noise_dim", C.c_int), ("f_T", _Mlp), ("f_Z", _Mlp), ("lik_obs", _Mlp),
                ("lik_state", _Mlp), ("lik_action_cond", C.c_int), ("lik_temperature", C.c_float),
                ("discount", C.c_float), ("reward", _Reward), ("prec", C.c_int),
                ("terminal", C.POINTER(_Terminal)), ("denoise_T", _Mlp), ("denoise_Z", _Mlp)]


def lib_path() -> str:
    return os.path.join(_HERE, "libvoila.so")


def load_library():
    """dlopen libvoila.so (building it in-tree first if it is missing or stale)."""
    global _LIB
    if _LIB is not None:
        return _LIB
    from . import build as _build
    path = _build.build()
    lib = C.CDLL(path)
    vp, i32, u64, sz = C.c_void_p, C.c_int, C.c_uint64, C.c_size_t
    lib.voila_create.argtypes = [C.POINTER(_ModelDesc), i32, C.POINTER(vp)]
    lib.voila_create.restype = i32
    lib.voila_destroy.argtypes = [vp]
    lib.voila_destroy.restype = None
    lib.voila_workspace_bytes.argtypes = [vp, i32, i32, i32, i32]
    lib.voila_workspace_bytes.restype = sz
    lib.voila_reserve.argtypes = [vp, i32, i32, i32, i32]
    lib.voila_reserve.restype = i32
    lib.voila_set_kernel.argtypes = [vp, i32]
    lib.voila_set_kernel.restype = i32
    lib.voila_tcgen05_supported.argtypes = [vp]
    lib.voila_tcgen05_supported.restype = i32
    lib.voila_rollout_values.argtypes = [vp, vp, i32, vp, i32, i32, vp, u64, vp, vp, vp, vp, vp]
    lib.voila_rollout_values.restype = i32
    lib.voila_belief_update.argtypes = [vp, vp, i32, C.c_int32, vp, vp, u64, vp, vp, vp, vp, vp, vp,
                                        vp, vp]
    lib.voila_belief_update.restype = i32
    lib.voila_belief_update_ess.argtypes = [vp, vp, i32, C.c_int32, vp, vp, u64, C.c_float, vp, vp, vp, vp, vp,
                                            vp, vp, vp, vp, vp]
    lib.voila_belief_update_ess.restype = i32
    lib.voila_resample_systematic.argtypes = [vp, vp, i32, u64, vp, vp, vp]
    lib.voila_resample_systematic.restype = i32
    lib.voila_resample_systematic_static.argtypes = [vp, i32, u64, vp, vp, vp]
    lib.voila_resample_systematic_static.restype = i32
    lib.voila_static_last_error.argtypes = []
    lib.voila_static_last_error.restype = C.c_char_p
    lib.voila_mlp_forward.argtypes = [vp, i32, vp, i32, vp, vp]
    lib.voila_mlp_forward.restype = i32
    lib.voila_best_action.argtypes = [vp, vp, vp, i32, i32, vp, vp, vp]
    lib.voila_best_action.restype = i32
    lib.voila_porpp_backup_level.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, C.c_float, C.c_float, vp, vp, vp]
    lib.voila_porpp_backup_level.restype = i32
    lib.voila_rollout_values_host.argtypes = [vp, vp, i32, vp, i32, i32, vp, u64, vp, vp, vp]
    lib.voila_rollout_values_host.restype = i32
    lib.voila_plan_host.argtypes = [vp, vp, i32, vp, i32, i32, vp, u64, vp, vp, vp, vp, vp]
    lib.voila_plan_host.restype = i32
    lib.voila_belief_update_host.argtypes = [vp, vp, i32, C.c_int32, vp, vp, u64, vp, vp, vp, vp, vp,
                                             vp]
    lib.voila_belief_update_host.restype = i32
    lib.voila_launch_count.argtypes = [vp]
    lib.voila_launch_count.restype = u64
    lib.voila_last_rollout_kernel.argtypes = [vp]
    lib.voila_last_rollout_kernel.restype = C.c_char_p
    lib.voila_last_belief_kernel.argtypes = [vp]
    lib.voila_last_belief_kernel.restype = C.c_char_p
    lib.voila_status_string.argtypes = [i32]
    lib.voila_status_string.restype = C.c_char_p
    lib.voila_last_cuda_error.argtypes = [vp]
    lib.voila_last_cuda_error.restype = C.c_char_p
    lib.voila_set_profiling.argtypes = [vp, i32]
    lib.voila_set_profiling.restype = i32
    lib.voila_profile_read.argtypes = [vp, i32, C.POINTER(C.c_float), i32]
    lib.voila_profile_read.restype = i32
    lib.voila_pw_workspace_bytes.argtypes = [vp, i32, i32, i32]
    lib.voila_pw_workspace_bytes.restype = sz
    lib.voila_pw_reserve.argtypes = [vp, i32, i32, i32]
    lib.voila_pw_reserve.restype = i32
    lib.voila_pw_update.argtypes = [vp, vp, i32, vp, i32, vp, vp, vp, vp, i32, C.c_double, C.c_double, vp, u64,
                                    vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.voila_pw_update.restype = i32
    lib.voila_porpp_backup.argtypes = [vp, C.POINTER(_PorppLevel), i32, i32, vp, C.c_float, C.c_float, vp, vp]
    lib.voila_porpp_backup.restype = i32
    lib.voila_diffusion_sample.argtypes = [vp, i32, vp, vp, i32, i32, u64, vp, vp]
    lib.voila_diffusion_sample.restype = i32
    lib.voila_version.argtypes = []
    lib.voila_version.restype = i32
    _LIB = lib
    return lib


def _fptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_float))


def _pack_mlp(f, keep: list) -> _Mlp:
    n = len(f.W)
    dims = (C.c_int * (n + 1))(*[int(d) for d in f.dims])
    Ws = [np.ascontiguousarray(w, dtype=np.float32) for w in f.W]
    bs = [np.ascontiguousarray(b, dtype=np.float32) for b in f.b]
    Wp = (C.POINTER(C.c_float) * n)(*[_fptr(w) for w in Ws])
    bp = (C.POINTER(C.c_float) * n)(*[_fptr(b) for b in bs])
    keep.extend([dims, Ws, bs, Wp, bp])
    return _Mlp(n, C.cast(dims, C.POINTER(C.c_int)), C.cast(Wp, C.POINTER(C.POINTER(C.c_float))),
                C.cast(bp, C.POINTER(C.POINTER(C.c_float))), int(f.act))


def _dptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _hptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr())


class Voila:
    """One libvoila context: packed generator / tower weights on one GPU plus a reserved workspace.

    `model` is duck-typed like synth.ModelSpec (S, O, A, Nz, f_T, f_Z, lik_obs, lik_state each
    with dims/act/W/b, lik_action_cond, lam, gamma, reward_kind, reward_param, action_cost, prec).
    All tensors passed to the device entry points are torch CUDA tensors on `device`.
    """

    def __init__(self, model, device: int = 0, prec: Optional[int] = None):
        import torch
        self._torch = torch
        self.lib = load_library()
        self.S, self.O, self.A, self.Nz = model.S, model.O, model.A, model.Nz
        self.prec = int(model.prec if prec is None else prec)
        self.device = int(device)
        self.d = int(model.lik_obs.dims[-1])
        keep: list = []
        desc = _ModelDesc()
        desc.state_dim, desc.obs_dim, desc.n_actions, desc.noise_dim = self.S, self.O, self.A, self.Nz
        desc.f_T = _pack_mlp(model.f_T, keep)
        desc.f_Z = _pack_mlp(model.f_Z, keep)
        desc.lik_obs = _pack_mlp(model.lik_obs, keep)
        desc.lik_state = _pack_mlp(model.lik_state, keep)
        desc.lik_action_cond = int(model.lik_action_cond)
        desc.lik_temperature = float(model.lam)
        desc.discount = float(model.gamma)
        param = np.ascontiguousarray(model.reward_param, dtype=np.float32).ravel()
        cost = None if model.action_cost is None else np.ascontiguousarray(model.action_cost, np.float32)
        keep.extend([param, cost])
        desc.reward = _Reward(int(model.reward_kind), _fptr(param), _fptr(cost))
        desc.prec = self.prec
        term = getattr(model, "terminal", None)
        if term is not None and len(term.radii):
            t_dims = np.asarray([len(c) for c in term.centers], dtype=np.int32)
            t_cen = np.concatenate([np.asarray(c, np.float32).ravel() for c in term.centers])
            t_rad = np.ascontiguousarray(term.radii, np.float32)
            t_rew = np.ascontiguousarray(term.rewards, np.float32)
            t_stop = np.ascontiguousarray(term.stops, np.int32)
            tstruct = _Terminal(len(t_dims), t_dims.ctypes.data_as(C.POINTER(C.c_int)), _fptr(t_cen),
                                _fptr(t_rad), _fptr(t_rew), t_stop.ctypes.data_as(C.POINTER(C.c_int)))
            keep.extend([t_dims, t_cen, t_rad, t_rew, t_stop, tstruct])
            desc.terminal = C.pointer(tstruct)
        for name in ("denoise_T", "denoise_Z"):
            f = getattr(model, name, None)
            if f is not None:
                setattr(desc, name, _pack_mlp(f, keep))
        h = C.c_void_p()
        self._h = None
        self._check(self.lib.voila_create(C.byref(desc), self.device, C.byref(h)), "voila_create")
        self._h = h
        self._res = (0, 0, 0, 0)

    # -- plumbing ------------------------------------------------------------------------------
    def _check(self, status: int, what: str):
        if status != 0:
            msg = self.lib.voila_status_string(status).decode()
            cuda = self.lib.voila_last_cuda_error(self._h).decode() if self._h else ""
            raise VoilaError(f"{what}: {msg}" + (f" ({cuda})" if cuda else ""))

    def close(self):
        if getattr(self, "_h", None):
            self.lib.voila_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def particle_dtype(self):
        return self._torch.bfloat16 if self.prec == PREC_BF16 else self._torch.float32

    def _stream(self):
        return C.c_void_p(self._torch.cuda.current_stream(self.device).cuda_stream)

    def voila_workspace_bytes(self, P, Q, H, N) -> int:
        return int(self.lib.voila_workspace_bytes(self._h, P, Q, H, N))

    def voila_reserve(self, P=0, Q=0, H=0, N=0):
        self._check(self.lib.voila_reserve(self._h, P, Q, H, N), "voila_reserve")
        self._res = (P, Q, H, N)

    def _ensure(self, P=0, Q=0, H=0, N=0):
        r = self._res
        if P > r[0] or Q > r[1] or H > r[2] or N > r[3]:
            self.voila_reserve(max(P, r[0]), max(Q, r[1]), max(H, r[2]), max(N, r[3]))

    def voila_set_kernel(self, kernel: int):
        self._check(self.lib.voila_set_kernel(self._h, kernel), "voila_set_kernel")

    def voila_tcgen05_supported(self) -> bool:
        return bool(self.lib.voila_tcgen05_supported(self._h))

    def voila_launch_count(self) -> int:
        return int(self.lib.voila_launch_count(self._h))

    def voila_last_belief_kernel(self) -> str:
        return self.lib.voila_last_belief_kernel(self._h).decode()

    def voila_last_rollout_kernel(self) -> str:
        return self.lib.voila_last_rollout_kernel(self._h).decode()

    def voila_set_profiling(self, on: bool):
        self._check(self.lib.voila_set_profiling(self._h, int(bool(on))), "voila_set_profiling")

    def voila_profile_read(self, which: int):
        buf = (C.c_float * 256)()
        n = self.lib.voila_profile_read(self._h, int(which), buf, 256)
        return [float(buf[i]) for i in range(n)]

    def to_particles(self, x: np.ndarray):
        """numpy fp32 [n][S] -> device tensor of the ctx's particle dtype (plain dtype conversion)."""
        t = self._torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(f"cuda:{self.device}")
        return t.to(self.particle_dtype).contiguous()

    # -- hot calls (device buffers) -------------------------------------------------------------
    def voila_rollout_values(self, particles, action_seqs, weights, seed, want_witness=True,
                             want_returns=False, want_final_states=False):
        torch = self._torch
        P, S = particles.shape
        Q, H = action_seqs.shape
        assert S == self.S and particles.dtype == self.particle_dtype and particles.is_contiguous()
        assert action_seqs.dtype == torch.int32 and action_seqs.is_contiguous()
        self._ensure(P=P, Q=Q, H=H)
        dev = particles.device
        values = torch.empty(Q, dtype=torch.float32, device=dev)
        witness = torch.empty((Q, self.O), dtype=torch.float32, device=dev) if want_witness else None
        returns = torch.empty((Q, P), dtype=torch.float32, device=dev) if want_returns else None
        finals = torch.empty((Q, P, S), dtype=torch.float32, device=dev) if want_final_states else None
        self._check(self.lib.voila_rollout_values(
            self._h, _dptr(particles), P, _dptr(action_seqs), Q, H, _dptr(weights),
            C.c_uint64(int(seed)), _dptr(values), _dptr(witness), _dptr(returns), _dptr(finals),
            self._stream()), "voila_rollout_values")
        out = {"values": values, "witness": witness}
        if want_returns:
            out["returns"] = returns
        if want_final_states:
            out["final_states"] = finals
        return out

    def belief_update_buffers(self, particles, want_debug=True):
        """Output buffers of voila_belief_update for particle sets shaped like `particles` (the caller
        may keep and reuse them: pass as `out=`; `out["particles"]` must not alias the input)."""
        torch = self._torch
        N = particles.shape[0]
        dev = particles.device
        out = {
            "particles": torch.empty_like(particles),
            "weights": torch.empty(N, dtype=torch.float32, device=dev),
            "ancestors": torch.empty(N, dtype=torch.int32, device=dev),
            "log_evidence": torch.empty(1, dtype=torch.float32, device=dev),
            "status": torch.empty(1, dtype=torch.int32, device=dev),
        }
        if want_debug:
            out["post_weights"] = torch.empty(N, dtype=torch.float32, device=dev)
            out["proposals"] = torch.empty_like(particles)
        return out

    def voila_belief_update(self, particles, action, observation, weights, seed, want_debug=True, out=None,
                            ess_threshold=None):
        """ess_threshold=None: always resample (voila_belief_update); a float: adaptive resampling
        (voila_belief_update_ess), outputs "ess" and "resampled" added."""
        torch = self._torch
        N, S = particles.shape
        assert S == self.S and particles.dtype == self.particle_dtype and particles.is_contiguous()
        assert observation.dtype == torch.float32 and observation.numel() == self.O
        self._ensure(N=N)
        if out is None:
            out = self.belief_update_buffers(particles, want_debug)
        if ess_threshold is None:
            self._check(self.lib.voila_belief_update(
                self._h, _dptr(particles), N, int(action), _dptr(observation), _dptr(weights),
                C.c_uint64(int(seed)), _dptr(out["particles"]), _dptr(out["weights"]),
                _dptr(out["ancestors"]), _dptr(out.get("post_weights")), _dptr(out.get("proposals")),
                _dptr(out["log_evidence"]), _dptr(out["status"]), self._stream()), "voila_belief_update")
            return out
        if "ess" not in out:
            out["ess"] = torch.empty(1, dtype=torch.float32, device=particles.device)
            out["resampled"] = torch.empty(1, dtype=torch.int32, device=particles.device)
        self._check(self.lib.voila_belief_update_ess(
            self._h, _dptr(particles), N, int(action), _dptr(observation), _dptr(weights),
            C.c_uint64(int(seed)), C.c_float(float(ess_threshold)), _dptr(out["particles"]), _dptr(out["weights"]),
            _dptr(out["ancestors"]), _dptr(out.get("post_weights")), _dptr(out.get("proposals")),
            _dptr(out["log_evidence"]), _dptr(out["ess"]), _dptr(out["resampled"]), _dptr(out["status"]),
            self._stream()), "voila_belief_update_ess")
        return out

    def voila_pw_update(self, particles, group_off, group_action, visit_count, branch_count, branch_obs, k_o,
                        alpha_o, weights, seed, want_debug=True):
        """Vectorised progressive widening with batched likelihood (include/voila.h).  visit_count,
        branch_count ([G] int32) and branch_obs ([G][M_max][O] fp32) are device tensors updated IN PLACE."""
        torch = self._torch
        N, S = particles.shape
        G, M_max = branch_obs.shape[0], branch_obs.shape[1]
        assert S == self.S and particles.dtype == self.particle_dtype and particles.is_contiguous()
        assert group_off.dtype == torch.int32 and group_off.numel() == G + 1 and group_action.dtype == torch.int32
        assert visit_count.dtype == torch.int32 and branch_count.dtype == torch.int32
        assert branch_obs.dtype == torch.float32 and branch_obs.is_contiguous() and branch_obs.shape[2] == self.O
        self._ensure(N=N)
        res = getattr(self, "_pw_res", (0, 0))
        if res[0] < N or res[1] < G * M_max:
            self._check(self.lib.voila_pw_reserve(self._h, N, G, M_max), "voila_pw_reserve")
            self._pw_res = (N, G * M_max)
        dev = particles.device
        out = {"particles": torch.empty_like(particles),
               "weights": torch.empty(N, dtype=torch.float32, device=dev),
               "ancestors": torch.empty(N, dtype=torch.int32, device=dev),
               "sim_branch": torch.empty(N, dtype=torch.int32, device=dev),
               "seg_status": torch.empty(G * M_max, dtype=torch.int32, device=dev)}
        if want_debug:
            out["opened"] = torch.empty(N, dtype=torch.int32, device=dev)
            out["post_weights"] = torch.empty(N, dtype=torch.float32, device=dev)
            out["proposals"] = torch.empty_like(particles)
        self._check(self.lib.voila_pw_update(
            self._h, _dptr(particles), N, _dptr(group_off), G, _dptr(group_action), _dptr(visit_count),
            _dptr(branch_count), _dptr(branch_obs), M_max, C.c_double(float(k_o)), C.c_double(float(alpha_o)),
            _dptr(weights), C.c_uint64(int(seed)), _dptr(out["particles"]), _dptr(out["weights"]),
            _dptr(out["ancestors"]), _dptr(out["sim_branch"]), _dptr(out.get("opened")),
            _dptr(out.get("post_weights")), _dptr(out.get("proposals")), _dptr(out["seg_status"]),
            self._stream()), "voila_pw_update")
        return out

    def voila_diffusion_sample(self, which, cond, actions, K, seed):
        """The diffusion teacher's DDIM-ODE sampler (include/voila.h): K denoiser calls per sample.
        which = 0 transition teacher (-> [N][S]), 1 observation teacher (-> [N][O]); fp32 output."""
        torch = self._torch
        N = cond.shape[0]
        assert cond.dtype == self.particle_dtype and cond.is_contiguous() and cond.shape[1] == self.S
        assert actions.dtype == torch.int32 and actions.numel() == N
        out = torch.empty((N, self.S if which == 0 else self.O), dtype=torch.float32, device=cond.device)
        self._check(self.lib.voila_diffusion_sample(self._h, int(which), _dptr(cond), _dptr(actions), N, int(K),
                                                    C.c_uint64(int(seed)), _dptr(out), self._stream()),
                    "voila_diffusion_sample")
        return out

    def voila_resample_systematic(self, v, seed):
        torch = self._torch
        N = v.numel()
        assert v.dtype == torch.float32 and v.is_contiguous()
        self._ensure(N=N)
        anc = torch.empty(N, dtype=torch.int32, device=v.device)
        status = torch.empty(1, dtype=torch.int32, device=v.device)
        self._check(self.lib.voila_resample_systematic(
            self._h, _dptr(v), N, C.c_uint64(int(seed)), _dptr(anc), _dptr(status), self._stream()),
            "voila_resample_systematic")
        return anc, status

    def voila_mlp_forward(self, which, x):
        torch = self._torch
        rows = x.shape[0]
        assert x.dtype == torch.float32 and x.is_contiguous()
        out_dim = [self.S, self.O, self.d, self.d][which]
        y = torch.empty((rows, out_dim), dtype=torch.float32, device=x.device)
        self._check(self.lib.voila_mlp_forward(self._h, which, _dptr(x), rows, _dptr(y), self._stream()),
                    "voila_mlp_forward")
        return y

    def voila_best_action(self, values, action_seqs):
        """-> (best_q, best_action) device int32 tensors of one element each."""
        torch = self._torch
        Q, H = action_seqs.shape
        assert values.dtype == torch.float32 and values.numel() == Q
        bq = torch.empty(1, dtype=torch.int32, device=values.device)
        ba = torch.empty(1, dtype=torch.int32, device=values.device)
        self._check(self.lib.voila_best_action(self._h, _dptr(values), _dptr(action_seqs), Q, H,
                                               _dptr(bq), _dptr(ba), self._stream()), "voila_best_action")
        return bq, ba

    def voila_porpp_backup(self, levels, leaf_values, eta, gamma, per_level_calls=False):
        """PORPP preference backup (Eq. 1) of a whole tree: `levels[d]` = dict of device tensors
        R, logpi0 [nb, A] fp32, child_off [nb*A+1] int32, child_idx int32, child_w fp32.  One
        voila_porpp_backup call for the tree (per_level_calls=True: one voila_porpp_backup_level call
        per level, deepest first).  -> (V, Psi, root_action): lists over depth, int32 [root beliefs]."""
        torch = self._torch
        D = len(levels)
        dev = levels[0]["R"].device
        A = levels[0]["R"].shape[1]
        V = [torch.empty(lv["R"].shape[0], dtype=torch.float32, device=dev) for lv in levels]
        Psi = [torch.empty(lv["R"].shape, dtype=torch.float32, device=dev) for lv in levels]
        opt = lambda t: _dptr(t if t is not None and t.numel() else None)
        raw = lambda t: None if t is None or not t.numel() else t.data_ptr()
        if per_level_calls:
            v_next = leaf_values
            for d in range(D - 1, -1, -1):
                lv = levels[d]
                nb = lv["R"].shape[0]
                self._check(self.lib.voila_porpp_backup_level(
                    self._h, _dptr(lv["R"]), _dptr(lv["logpi0"]), _dptr(lv["child_off"]), opt(lv["child_idx"]),
                    opt(lv["child_w"]), opt(v_next), nb, A, C.c_float(eta), C.c_float(gamma), _dptr(Psi[d]),
                    _dptr(V[d]), self._stream()), "voila_porpp_backup_level")
                v_next = V[d]
            return V, Psi, None
        arr = (_PorppLevel * D)()
        for d, lv in enumerate(levels):
            arr[d] = _PorppLevel(raw(lv["R"]), raw(lv["logpi0"]), raw(lv["child_off"]), raw(lv["child_idx"]),
                                 raw(lv["child_w"]), int(lv["R"].shape[0]), raw(Psi[d]), raw(V[d]))
        root = torch.empty(levels[0]["R"].shape[0], dtype=torch.int32, device=dev)
        self._check(self.lib.voila_porpp_backup(self._h, arr, D, A, opt(leaf_values), C.c_float(eta), C.c_float(gamma),
                                                _dptr(root), self._stream()), "voila_porpp_backup")
        return V, Psi, root

    # -- host-buffer variants (pinned torch CPU tensors or numpy arrays) --------------------------
    def voila_rollout_values_host(self, particles, action_seqs, weights, seed, values_out,
                                  witness_out=None):
        P, Q, H = particles.shape[0], action_seqs.shape[0], action_seqs.shape[1]
        self._ensure(P=P, Q=Q, H=H)
        self._check(self.lib.voila_rollout_values_host(
            self._h, _hptr(particles), P, _hptr(action_seqs), Q, H, _hptr(weights),
            C.c_uint64(int(seed)), _hptr(values_out), _hptr(witness_out), self._stream()),
            "voila_rollout_values_host")
        return values_out

    def voila_plan_host(self, particles, action_seqs, weights, seed, values_out, best_out, witness_out=None):
        """Rollout + executed action through host buffers; best_out: host int32 [2] = (q*, first action)."""
        P, Q, H = particles.shape[0], action_seqs.shape[0], action_seqs.shape[1]
        self._ensure(P=P, Q=Q, H=H)
        bq = _hptr(best_out)
        ba = C.c_void_p(bq.value + 4)
        self._check(self.lib.voila_plan_host(
            self._h, _hptr(particles), P, _hptr(action_seqs), Q, H, _hptr(weights), C.c_uint64(int(seed)),
            _hptr(values_out), _hptr(witness_out), bq, ba, self._stream()), "voila_plan_host")
        return values_out

    def voila_belief_update_host(self, particles, action, observation, weights, seed, particles_out,
                                 weights_out=None, ancestors_out=None, log_evidence_out=None,
                                 status_out=None):
        N = particles.shape[0]
        self._ensure(N=N)
        self._check(self.lib.voila_belief_update_host(
            self._h, _hptr(particles), N, int(action), _hptr(observation), _hptr(weights),
            C.c_uint64(int(seed)), _hptr(particles_out), _hptr(weights_out), _hptr(ancestors_out),
            _hptr(log_evidence_out), _hptr(status_out), self._stream()), "voila_belief_update_host")
        return particles_out
