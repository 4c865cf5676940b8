#!/usr/bin/env python
"""bench.py -- one planning step of VOiLA's hot path on synthetic, seeded inputs.

A "step" is one pass of the whole hot path over one batch: voila_rollout_values on P particles x
Q action sequences x horizon H, then voila_belief_update on N particles (SURVEY.md 8(a) rows
R1-R11).  metric = rollout steps/s = P*Q*H*n_gpus / step time, with the belief-update latency and
per-kernel times alongside.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl voila|reference]

Multi-GPU (torchrun): the path does not shard (north_star: one GPU, no collectives) -> every rank
runs an independent replica ("replicas only"); value = units of all ranks / max time.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

DEFAULT_CONFIG = 5  # the largest config: the one north_star's >= 50 %-of-peak target is stated on
METRIC = "rollout_steps_per_sec"
UNIT = "particle*sequence*depth steps/s"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_burst": d["bf16_tflops"],
                "bf16_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]), "src": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "src": "fallback"}


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        super().__init__(daemon=True)
        self.index = index
        self.rows = []
        self.stop_flag = False
        self.proc = None

    def run(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append(line.strip())
                if self.stop_flag:
                    break
        except Exception:
            pass

    def finish(self):
        self.stop_flag = True
        if self.proc is not None:
            try:
                self.proc.terminate()
            except Exception:
                pass
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown",
                                "sw_power_cap"], f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)),
                "reasons": sorted(reasons), "samples": len(sm)}


def _flops_fp32_peak_tflops(sm_count, sm_mhz):
    # 4 SMSPs x 32 FFMA lanes x 2 flop per SM per clock (B300_MICROARCH.md "Pipe rates")
    return sm_count * 128 * 2 * sm_mhz * 1e6 / 1e12


def _oracle_sample(cfg, model, inp, target_s=12.0):
    """Times the oracle (as it stands) on a bounded sample of the workload: all P particles x Q'
    sequences x H plus a belief update on N*Q'/Q particles; returns (steps/s, cores, description)."""
    from oracle import voila_oracle as oracle
    from paper_2606_19729_b200 import synth
    bf16 = model.prec == synth.PREC_BF16
    parts = synth.bf16_round_np(inp.particles) if bf16 else inp.particles
    bu_parts = synth.bf16_round_np(inp.bu_particles) if bf16 else inp.bu_particles
    om = oracle.OracleModel(model)
    cores = oracle.num_threads()
    P, (Q, H) = parts.shape[0], inp.action_seqs.shape
    # probe: one sequence per thread on a particle subset
    Pp = min(P, 64)
    qp = min(Q, cores)
    t0 = time.perf_counter()
    om.rollout_values(parts[:Pp], inp.action_seqs[:qp], None, 1)
    dt = max(time.perf_counter() - t0, 1e-4)
    rate = Pp * qp * H / dt
    want = rate * target_s
    Ps = P if want >= P * H * qp else max(Pp, int(want / (H * qp)))
    Qs = int(min(Q, max(qp, (want / (Ps * H)) // qp * qp)))
    Ns = max(1, int(round(bu_parts.shape[0] * (Ps * Qs) / (P * Q))))
    t0 = time.perf_counter()
    om.rollout_values(parts[:Ps], inp.action_seqs[:Qs], None, 1)
    om.belief_update(bu_parts[:Ns], inp.bu_action, inp.observation,
                     None if inp.bu_weights is None else inp.bu_weights[:Ns], 2)
    dt = time.perf_counter() - t0
    desc = (f"{Ps} of {P} particles x {Qs} of {Q} sequences x H={H} rollout + belief update on "
            f"{Ns} of {bu_parts.shape[0]} particles, {dt:.1f} s")
    return Ps * Qs * H / dt, cores, desc, dt


def _oracle_one_thread(cfg, model, inp, target_s=2.0):
    """The oracle on ONE host thread (SURVEY 8d asks for both figures): a small rollout slice."""
    from oracle import voila_oracle as oracle
    from paper_2606_19729_b200 import synth
    parts = synth.bf16_round_np(inp.particles) if model.prec == synth.PREC_BF16 else inp.particles
    om = oracle.OracleModel(model)
    n = oracle.num_threads()
    oracle.set_num_threads(1)
    try:
        H = inp.action_seqs.shape[1]
        Pp = min(parts.shape[0], 16)
        t0 = time.perf_counter()
        om.rollout_values(parts[:Pp], inp.action_seqs[:1], None, 1)
        dt = max(time.perf_counter() - t0, 1e-4)
        Ps = int(min(parts.shape[0], max(Pp, Pp * target_s / dt)))
        t0 = time.perf_counter()
        om.rollout_values(parts[:Ps], inp.action_seqs[:1], None, 1)
        dt = time.perf_counter() - t0
        return Ps * H / dt
    finally:
        oracle.set_num_threads(n)


def _porpp_leg(ctx, dev, peaks):
    """the PORPP preference backup (Eq. 1) on a wide synthetic level: 2^18 belief nodes x
    16 actions x 4 observation branches, the children numbered in creation order as the tree tensors
    grow (every belief node of the next level has exactly one parent), plus the same level with
    scattered child indices (a worst case no tree produces).  One voila_porpp_backup call each."""
    import torch
    nb, A, B = 1 << 18, 16, 4
    na = nb * A
    g = torch.Generator(device=dev)
    g.manual_seed(20260619)
    lv = dict(R=torch.randn((nb, A), generator=g, device=dev),
              logpi0=torch.full((nb, A), -float(np.log(A)), device=dev),
              child_off=torch.arange(0, na * B + 1, B, dtype=torch.int32, device=dev),
              child_idx=torch.arange(0, na * B, dtype=torch.int32, device=dev),
              child_w=torch.full((na * B,), 1.0 / B, device=dev))
    leaves = torch.randn(na * B, generator=g, device=dev)
    out = {}
    for name in ("tree", "scattered"):
        if name == "scattered":
            lv = dict(lv, child_idx=torch.randint(0, 1 << 20, (na * B,), generator=g, device=dev, dtype=torch.int32))
        for _ in range(3):
            ctx.voila_porpp_backup([lv], leaves, 2.0, 0.95)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        a.record()
        for _ in range(10):
            ctx.voila_porpp_backup([lv], leaves, 2.0, 0.95)
        b.record()
        torch.cuda.synchronize(dev)
        ms = a.elapsed_time(b) / 10
        # R, log pi0, row offset, Psi out per action node; index + weight (+ V(child), read once in a tree) per
        # branch; V and the root action out per belief node
        per_branch = 12 if name == "tree" else 8
        bytes_alg = na * 16 + na * B * per_branch + nb * 8
        gbs = bytes_alg / (ms * 1e-3) / 1e9
        out[name] = {"latency_us": 1e3 * ms,
                     "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                  "frac": gbs / peaks["hbm_gbs"], "bytes_per_action_node": bytes_alg / na}}
    out["scattered"]["roofline"]["note"] = ("child indices drawn at random over 2^20 nodes: 4-byte gathers cost a "
                                            "32-byte L2 sector each; V(child) is L2-resident and not counted")
    return {"workload": f"{nb} belief nodes x {A} actions x {B} branches, one level, root action",
            "latency_us": out["tree"]["latency_us"], "roofline": out["tree"]["roofline"],
            "scattered_children": out["scattered"]}


def _belief_roofs(N, row_bytes, kt, flop_particle, peaks, belief_kernel, unique_frac=None):
    """Sub-rooflines of one belief update from the library's per-kernel event pairs (ms lists)."""
    out = {}
    if kt[1] and "belief_tc2" in belief_kernel:
        tf = N * flop_particle / (np.mean(kt[1]) * 1e-3) / 1e12
        out["propose_score_roofline"] = {"bound": "tensor", "achieved": tf, "peak": peaks["bf16_burst"],
                                         "unit": "TFLOP/s", "frac": tf / peaks["bf16_burst"],
                                         "kernel": belief_kernel, "flop_per_particle": flop_particle}
    if kt[2]:
        b = N * (4 + 8)  # logit read, CDF write
        gbs = b / (np.mean(kt[2]) * 1e-3) / 1e9
        out["scan_roofline"] = {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                "frac": gbs / peaks["hbm_gbs"], "bytes_per_particle": 12}
    if kt[3]:
        # CDF read 8, row gather, row write, index 4, weight 4.  SURVEY 8(d) also states the count with
        # only the DISTINCT ancestor rows read (u = measured fraction of distinct ancestors).
        b = N * (8 + 2 * row_bytes + 8)
        gbs = b / (np.mean(kt[3]) * 1e-3) / 1e9
        r = {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
             "frac": gbs / peaks["hbm_gbs"], "bytes_per_particle": 8 + 2 * row_bytes + 8}
        if unique_frac is not None:
            bu = 8 + row_bytes * unique_frac + row_bytes + 8
            gu = N * bu / (np.mean(kt[3]) * 1e-3) / 1e9
            r.update({"unique_ancestor_frac": unique_frac, "bytes_per_particle_unique_rows": bu,
                      "achieved_unique_rows": gu, "frac_unique_rows": gu / peaks["hbm_gbs"]})
        out["resample_roofline"] = r
    for r in out.values():
        nominal = 2250.0 if r["bound"] == "tensor" else 8000.0
        r["nominal_peak"] = nominal
        r["frac_of_nominal"] = r["achieved"] / nominal
    return out


def _leg_belief_cfg4(vl, synth, dev, local, peaks, flush, calls=20):
    """The belief-update half of the metric at the size it is defined on (BASELINE.json config 4:
    2^20 particles, skewed prior weights): >= 20 timed calls, L2 flushed between calls, CUDA events
    on the launching stream; per-kernel times from the library's event pairs; e2e through
    voila_belief_update_host (pinned host buffers, copies inside the timed region)."""
    import torch
    cfg = synth.CONFIGS[4]
    model = synth.make_model(cfg)
    inp = synth.make_inputs(cfg)
    N = cfg.N
    ctx = vl.Voila(model, device=local)
    ctx.voila_reserve(0, 0, 0, N)
    parts = ctx.to_particles(inp.bu_particles)
    obs = torch.from_numpy(inp.observation).to(dev)
    w = torch.from_numpy(inp.bu_weights).to(dev)
    bufs = ctx.belief_update_buffers(parts, want_debug=False)
    stream = torch.cuda.current_stream(dev)
    for k in range(3):
        ctx.voila_belief_update(parts, inp.bu_action, obs, w, 7000 + k, want_debug=False, out=bufs)
    torch.cuda.synchronize(dev)
    ctx.voila_set_profiling(True)
    for which in range(4):
        ctx.voila_profile_read(which)
    l0 = ctx.voila_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(calls)]
    for k in range(calls):
        flush.fill_(k & 0xFF)
        ev[k][0].record(stream)
        ctx.voila_belief_update(parts, inp.bu_action, obs, w, 7100 + k, want_debug=False, out=bufs)
        ev[k][1].record(stream)
    torch.cuda.synchronize(dev)
    launches = ctx.voila_launch_count() - l0
    ms = [a.elapsed_time(b) for a, b in ev]
    kt = [ctx.voila_profile_read(which) for which in range(4)]
    ctx.voila_set_profiling(False)
    assert int(bufs["status"].item()) == 0
    uniq = float(torch.unique(bufs["ancestors"]).numel()) / N  # measurement only (distinct ancestor rows)
    row = cfg.S * 2
    leg = {"workload": f"{cfg.name}: N={N} particles, prior log-weights ~ N(0,4)", "calls": calls,
           "latency_us": 1e3 * float(np.mean(ms)), "latency_us_best": 1e3 * float(np.min(ms)),
           "particles_per_s": N / (float(np.mean(ms)) * 1e-3),
           "propose_score_us": 1e3 * float(np.mean(kt[1])) if kt[1] else None,
           "scan_us": 1e3 * float(np.mean(kt[2])) if kt[2] else None,
           "resample_gather_us": 1e3 * float(np.mean(kt[3])) if kt[3] else None,
           "gpu_launches_per_call": launches / calls, "l2": "flushed between calls (256 MiB write)"}
    leg.update(_belief_roofs(N, row, kt, synth.flops_per_belief_particle(model), peaks,
                             ctx.voila_last_belief_kernel(), unique_frac=uniq))
    # end to end: host buffers in, resampled particles + ancestors out
    h_p = parts.cpu().pin_memory()
    h_w = w.cpu().pin_memory()
    h_o = obs.cpu().pin_memory()
    h_out = torch.empty_like(h_p).pin_memory()
    h_anc = torch.empty(N, dtype=torch.int32).pin_memory()
    h_le = torch.empty(1, dtype=torch.float32).pin_memory()
    h_st = torch.empty(1, dtype=torch.int32).pin_memory()
    ctx.voila_belief_update_host(h_p, inp.bu_action, h_o, h_w, 7200, h_out, None, h_anc, h_le, h_st)
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    n_e2e = 5
    for k in range(n_e2e):
        ctx.voila_belief_update_host(h_p, inp.bu_action, h_o, h_w, 7201 + k, h_out, None, h_anc, h_le, h_st)
    torch.cuda.synchronize(dev)
    dt = (time.perf_counter() - t0) / n_e2e
    leg["e2e"] = {"latency_us": 1e6 * dt, "particles_per_s": N / dt, "api": "voila_belief_update_host",
                  "h2d_bytes_per_call": N * row + N * 4 + cfg.O * 4, "d2h_bytes_per_call": N * row + N * 4 + 8}
    ctx.close()
    return leg


def _leg_rollout_cfg3(vl, synth, dev, local, peaks, flush, calls=5):
    """The rollout on the paper-shaped config (BASELINE.json config 3: 48-dim state, 256-wide
    generators; PAPER.md:165, :171 give 39-45-dim states): full size, L2 flushed between calls."""
    import torch
    cfg = synth.CONFIGS[3]
    model = synth.make_model(cfg)
    inp = synth.make_inputs(cfg)
    ctx = vl.Voila(model, device=local)
    ctx.voila_reserve(cfg.P, cfg.Q, cfg.H, 0)
    parts = ctx.to_particles(inp.particles)
    seqs = torch.from_numpy(inp.action_seqs).to(dev)
    for k in range(3):
        ctx.voila_rollout_values(parts, seqs, None, 8000 + k)
    torch.cuda.synchronize(dev)
    ctx.voila_set_profiling(True)
    ctx.voila_profile_read(0)
    stream = torch.cuda.current_stream(dev)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(calls)]
    for k in range(calls):
        flush.fill_(k & 0xFF)
        ev[k][0].record(stream)
        out = ctx.voila_rollout_values(parts, seqs, None, 8100 + k)
        ev[k][1].record(stream)
    torch.cuda.synchronize(dev)
    ms = [a.elapsed_time(b) for a, b in ev]
    kt = ctx.voila_profile_read(0)
    ctx.voila_set_profiling(False)
    assert bool(torch.isfinite(out["values"]).all())
    units = cfg.P * cfg.Q * cfg.H
    flop = synth.flops_per_rollout_step(model, algorithmic=True)
    k_ms = float(np.mean(kt)) if kt else float(np.mean(ms))
    tf = units * flop / (k_ms * 1e-3) / 1e12
    leg = {"workload": f"{cfg.name}: P={cfg.P} Q={cfg.Q} H={cfg.H}", "calls": calls,
           "rollout_ms": float(np.mean(ms)), "value": units / (float(np.mean(ms)) * 1e-3), "unit": UNIT,
           "roofline": {"bound": "tensor", "achieved": tf, "peak": peaks["bf16_burst"], "unit": "TFLOP/s",
                        "frac": tf / peaks["bf16_burst"], "kernel": ctx.voila_last_rollout_kernel(),
                        "kernel_ms": k_ms, "flop_per_unit": flop, "units_per_launch": units,
                        "nominal_peak": 2250.0, "frac_of_nominal": tf / 2250.0,
                        "peak_kind": f"bf16 burst, {peaks['src']}"}}
    ctx.close()
    return leg


def _leg_pw(vl, synth, dev, local, peaks, flush, calls=10):
    """vectorised progressive widening with batched likelihood on the
    quadruped-shaped model (config 3): 2^18 parallel simulations grouped under 2048 action nodes of
    ragged size, up to 16 observation branches per node, half of them open before the call."""
    import torch
    cfg = synth.CONFIGS[3]
    model = synth.make_model(cfg)
    N, G, M = 1 << 18, 2048, 16
    rng = np.random.default_rng(20260619 + 77)
    parts_np = rng.standard_normal((N, cfg.S)).astype(np.float32)
    cuts = np.concatenate([[0], np.sort(rng.integers(0, N + 1, G - 1)), [N]]).astype(np.int32)
    acts = rng.integers(0, cfg.A, G).astype(np.int32)
    bc0 = rng.integers(0, M // 2 + 1, G).astype(np.int32)
    vc0 = (bc0 * 8).astype(np.int32)
    bo0 = rng.standard_normal((G, M, cfg.O)).astype(np.float32)
    ctx = vl.Voila(model, device=local)
    parts = ctx.to_particles(parts_np)
    t = lambda a: torch.from_numpy(a).to(dev)
    go, ga = t(cuts), t(acts)

    def call(k):
        return ctx.voila_pw_update(parts, go, ga, t(vc0), t(bc0), t(bo0), 1.5, 0.5, None, 9000 + k, want_debug=False)

    for k in range(3):
        out = call(k)
    torch.cuda.synchronize(dev)
    ctx.voila_set_profiling(True)
    ctx.voila_profile_read(1)
    l0 = ctx.voila_launch_count()
    stream = torch.cuda.current_stream(dev)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(calls)]
    for k in range(calls):
        vc, bc, bo = t(vc0), t(bc0), t(bo0)
        flush.fill_(k & 0xFF)
        ev[k][0].record(stream)
        out = ctx.voila_pw_update(parts, go, ga, vc, bc, bo, 1.5, 0.5, None, 9100 + k, want_debug=False)
        ev[k][1].record(stream)
    torch.cuda.synchronize(dev)
    ms = [a.elapsed_time(b) for a, b in ev]
    kt = ctx.voila_profile_read(1)
    launches = (ctx.voila_launch_count() - l0) / calls
    ctx.voila_set_profiling(False)
    assert int(out["seg_status"].sum().item()) == 0
    flop = synth.flops_per_belief_particle(model)
    leg = {"workload": f"{N} simulations, {G} action nodes (ragged), M_max={M}, config-3 model",
           "latency_us": 1e3 * float(np.mean(ms)), "simulations_per_s": N / (float(np.mean(ms)) * 1e-3),
           "branches_opened": int((bc.cpu().numpy() - bc0).sum()), "gpu_launches_per_call": launches,
           "propose_score_us": 1e3 * float(np.mean(kt)) if kt else None, "kernel": ctx.voila_last_belief_kernel()}
    if kt and "belief_tc2" in ctx.voila_last_belief_kernel():
        tf = N * flop / (np.mean(kt) * 1e-3) / 1e12
        leg["propose_score_roofline"] = {"bound": "tensor", "achieved": tf, "peak": peaks["bf16_burst"],
                                         "unit": "TFLOP/s", "frac": tf / peaks["bf16_burst"],
                                         "flop_per_simulation": flop, "nominal_peak": 2250.0,
                                         "frac_of_nominal": tf / 2250.0}
    ctx.close()
    return leg


def _leg_diffusion(vl, synth, dev, local, peaks, K=32, N=1 << 16):
    """the diffusion teacher's sampler next to the distilled generator it is distilled into
    (PAPER.md:202 reports 8.6e5 / 1.2e6 samples/s distilled vs 8.2e3 / 1.8e4 for the diffusion models at
    batch 1024 on a laptop GPU, "up to 105x"): config-3 shapes, denoisers 4 x 512 SiLU, K = 32 DDIM-ODE
    steps, against the f_T proposals of one belief update of the same batch (propose + score kernel)."""
    import torch
    cfg = synth.CONFIGS[3]
    vT, vZ = synth.make_denoisers(cfg, [512, 512, 512, 512])
    model = synth.make_model(cfg).replace(denoise_T=vT, denoise_Z=vZ)
    rng = np.random.default_rng(20260619 + 88)
    ctx = vl.Voila(model, device=local)
    cond = ctx.to_particles(rng.standard_normal((N, cfg.S)).astype(np.float32))
    act = torch.from_numpy(rng.integers(0, cfg.A, N).astype(np.int32)).to(dev)
    out = {}
    for which, name in ((0, "transition"), (1, "observation")):
        for _ in range(2):
            ctx.voila_diffusion_sample(which, cond, act, K, 1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        a.record()
        for r in range(3):
            ctx.voila_diffusion_sample(which, cond, act, K, 2 + r)
        b.record()
        torch.cuda.synchronize(dev)
        ms = a.elapsed_time(b) / 3
        f = vT if which == 0 else vZ
        flop = 2 * sum(f.dims[l] * f.dims[l + 1] for l in range(len(f.W))) * K
        out[name] = {"samples_per_s": N / (ms * 1e-3), "ms": ms, "denoiser_calls": K,
                     "tflops": N * flop / (ms * 1e-3) / 1e12, "kernel": ctx.voila_last_belief_kernel() or "diffusion_step_ffma_kernel"}
    # the distilled side: one f_T sample per particle inside the belief update's propose+score kernel
    obs = torch.zeros(cfg.O, device=dev)
    bufs = ctx.belief_update_buffers(cond, want_debug=False)
    ctx.voila_set_profiling(True)
    for _ in range(3):
        ctx.voila_belief_update(cond, 1, obs, None, 5, want_debug=False, out=bufs)
    torch.cuda.synchronize(dev)
    ctx.voila_profile_read(1)
    for _ in range(5):
        ctx.voila_belief_update(cond, 1, obs, None, 6, want_debug=False, out=bufs)
    torch.cuda.synchronize(dev)
    kt = ctx.voila_profile_read(1)
    ctx.voila_set_profiling(False)
    dist = N / (float(np.mean(kt)) * 1e-3)
    ctx.close()
    return {"workload": f"{N} samples, config-3 shapes, denoisers 4x512, K={K}", "teacher": out,
            "distilled_f_T_samples_per_s": dist, "distilled_note": "f_T proposal + state tower + score per sample "
            "(the belief update's propose+score kernel): an upper bound on the cost of one f_T sample",
            "ratio_transition": dist / out["transition"]["samples_per_s"],
            "paper": "PAPER.md:202: 8.6e5 vs 8.2e3 (transition), 1.2e6 vs 1.8e4 (observation) samples/s, up to 105x, laptop RTX 3500 Ada"}


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    from paper_2606_19729_b200 import synth
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = synth.CONFIGS[args.config]
    model = synth.make_model(cfg)
    inp = synth.make_inputs(cfg)
    n = args.warmup + args.steps
    per = max(2.0, min(20.0, 150.0 / n))
    vals, times, desc, cores = [], [], "", 0
    for i in range(n):
        v, cores, desc, dt = _oracle_sample(cfg, model, inp, target_s=per)
        if i >= args.warmup:
            vals.append(v)
            times.append(dt)
    value = float(np.mean(vals))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "P": cfg.P, "Q": cfg.Q, "H": cfg.H, "N": cfg.N,
                   "note": "each step is a bounded sample of the workload (see cpu_baseline.sample)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_voila(args):
    import torch

    import paper_2606_19729_b200 as vl
    from paper_2606_19729_b200 import synth

    from paper_2606_19729_b200 import replicas
    rank, local, world = replicas.env_rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = torch.device(f"cuda:{local}")
    cfg = synth.CONFIGS[args.config]
    model = synth.make_model(cfg)
    inp = synth.make_inputs(cfg)
    P, Q, H, N = args.P or cfg.P, args.Q or cfg.Q, args.H or cfg.H, args.N or cfg.N
    reduced = (P, Q, H, N) != (cfg.P, cfg.Q, cfg.H, cfg.N)
    inp = synth.make_inputs(cfg, P=P, Q=Q, H=H, N=N)
    ctx = vl.Voila(model, device=local)
    if args.kernel != "auto":
        ctx.voila_set_kernel(vl.KERNEL_FFMA if args.kernel == "ffma" else vl.KERNEL_TCGEN05)
    ctx.voila_reserve(P, Q, H, N)
    chain = N == P  # the belief update's output particles are the next step's rollout particles
    parts = ctx.to_particles(inp.particles)
    bu_parts = parts if chain else ctx.to_particles(inp.bu_particles)
    seqs = torch.from_numpy(inp.action_seqs).to(dev)
    # one observation per planning step; rows padded to 16 bytes (the C ABI wants aligned pointers)
    obs_np = synth.observations_for_steps(cfg, args.warmup + args.steps + 1)
    o_pad = (cfg.O + 3) // 4 * 4
    obs_buf = torch.zeros(obs_np.shape[0], o_pad, dtype=torch.float32, device=dev)
    obs_buf[:, :cfg.O] = torch.from_numpy(obs_np).to(dev)
    obs_all = [obs_buf[k, :cfg.O] for k in range(obs_np.shape[0])]
    bu_w = None if inp.bu_weights is None else torch.from_numpy(inp.bu_weights).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2
    stream = torch.cuda.current_stream(dev)
    seed0 = replicas.replica_seed(20260619, rank, 0, 0)  # replicas draw different noise

    state = {"parts": parts, "bu_parts": bu_parts}
    # belief-update outputs are allocated once and reused (two sets: the chained configs feed the
    # resampled particles back in, and the output must not alias the input)
    bu_bufs = [ctx.belief_update_buffers(bu_parts, want_debug=False) for _ in range(2)]

    def pick_action(values):
        """CFG5 protocol: the executed action is the first action of argmax_q V_q, taken
        on the device (`voila_best_action`); the 4-byte read-back is the planner's output.  CFG1-4
        update with the fixed action of the config."""
        if cfg.index != 5:
            return inp.bu_action
        _, ba = ctx.voila_best_action(values, seqs)
        return int(ba.item())

    def step(k):
        out = ctx.voila_rollout_values(state["parts"], seqs, None, seed0 + 2 * k, want_witness=True)
        bu = ctx.voila_belief_update(state["bu_parts"], pick_action(out["values"]), obs_all[k], bu_w,
                                     seed0 + 2 * k + 1, want_debug=False, out=bu_bufs[k & 1])
        if chain:
            state["parts"] = state["bu_parts"] = bu["particles"]
        return out, bu

    for k in range(args.warmup):
        step(k)
    torch.cuda.synchronize(dev)
    ctx.voila_set_profiling(True)
    for w in range(4):
        ctx.voila_profile_read(w)
    launches0 = ctx.voila_launch_count()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
        time.sleep(0.25)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(dev)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True),
           torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for k in range(args.steps):
        flush.fill_(k & 0xFF)  # evict L2 between timed iterations (outside the event pairs)
        ev[k][0].record(stream)
        out = ctx.voila_rollout_values(state["parts"], seqs, None, seed0 + 2 * (k + args.warmup))
        a_exec = pick_action(out["values"])  # planning ends with the executed action (CFG5: 4-byte read-back)
        ev[k][1].record(stream)
        bu = ctx.voila_belief_update(state["bu_parts"], a_exec, obs_all[k + args.warmup], bu_w,
                                     seed0 + 2 * (k + args.warmup) + 1, want_debug=False,
                                     out=bu_bufs[(k + args.warmup) & 1])
        ev[k][2].record(stream)
        if chain:
            state["parts"] = state["bu_parts"] = bu["particles"]
    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    clocks = sampler.finish() if sampler else None
    launches = ctx.voila_launch_count() - launches0
    roll_ms = [a.elapsed_time(b) for a, b, _ in ev]
    bu_ms = [b.elapsed_time(c) for _, b, c in ev]
    total_ms = float(sum(roll_ms) + sum(bu_ms))
    total_ms = replicas.max_over_ranks(total_ms, dist, dev)  # the job is as slow as its slowest replica
    kt = [ctx.voila_profile_read(w) for w in range(4)]
    ctx.voila_set_profiling(False)
    assert int(bu["status"].item()) == 0 and bool(torch.isfinite(out["values"]).all())
    # belief updates issued back to back (no host synchronisation, no profiling events, L2 warm): the
    # per-call time once the host-side cost of issuing a call (Python + 4 launches) overlaps the kernels of
    # the call before; the timed-loop latency above starts from an idle GPU right after a host read-back
    n_b2b = 50
    b2b = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
    src, a_b2b = state["bu_parts"].clone(), (inp.bu_action if cfg.index != 5 else 0)
    for _ in range(3):
        ctx.voila_belief_update(src, a_b2b, obs_all[0], bu_w, 4242, want_debug=False, out=bu_bufs[0])
    torch.cuda.synchronize(dev)
    b2b[0].record(stream)
    for i in range(n_b2b):
        ctx.voila_belief_update(src, a_b2b, obs_all[0], bu_w, 4243 + i, want_debug=False, out=bu_bufs[i & 1])
    b2b[1].record(stream)
    torch.cuda.synchronize(dev)
    bu_b2b_us = 1e3 * b2b[0].elapsed_time(b2b[1]) / n_b2b
    ms_per_step = total_ms / args.steps
    value = replicas.whole_job_value(P * Q * H, world, ms_per_step)

    # ---- end to end through the host-buffer C-ABI entry points (pinned host memory) ----
    esize = 2 if ctx.prec == vl.PREC_BF16 else 4
    h_parts = parts.cpu().pin_memory()
    h_bu = h_parts if chain else bu_parts.cpu().pin_memory()
    h_seqs = torch.from_numpy(inp.action_seqs).pin_memory()
    h_obs = obs_buf.cpu().pin_memory()
    h_w = None if bu_w is None else bu_w.cpu().pin_memory()
    h_vals = torch.empty(Q, dtype=torch.float32).pin_memory()
    h_pout = torch.empty_like(h_bu).pin_memory()
    h_anc = torch.empty(N, dtype=torch.int32).pin_memory()
    h_le = torch.empty(1, dtype=torch.float32).pin_memory()
    h_st = torch.empty(1, dtype=torch.int32).pin_memory()
    e2e_steps = max(1, min(args.steps, 3))

    h_best = torch.zeros(2, dtype=torch.int32).pin_memory()

    def e2e_step(k):
        # planning half through the C ABI: rollout + executed action (argmax on the device), host buffers
        ctx.voila_plan_host(h_parts, h_seqs, None, seed0 + 2 * k, h_vals, h_best)
        a_exec = int(h_best[1]) if cfg.index == 5 else inp.bu_action
        ctx.voila_belief_update_host(h_bu, a_exec, h_obs[k % h_obs.shape[0], :cfg.O], h_w,
                                     seed0 + 2 * k + 1, h_pout, None, h_anc, h_le, h_st)

    e2e_step(0)
    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        e2e_step(k + 1)
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0
    e2e_s = replicas.max_over_ranks(e2e_s, dist, dev)
    h2d = P * cfg.S * esize + Q * H * 4 + N * cfg.S * esize + cfg.O * 4 + (N * 4 if h_w is not None else 0)
    d2h = Q * 4 + 8 + N * cfg.S * esize + N * 4 + 8
    e2e = {"value": world * P * Q * H * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "steps": e2e_steps,
           "api": "voila_plan_host + voila_belief_update_host"}
    if rank != 0:
        return

    # ---- roofline of the dominant kernel (the rollout kernel), from the library's event pairs ----
    peaks = _peaks()
    flop_step = synth.flops_per_rollout_step(model, algorithmic=True)
    k_ms = float(np.mean(kt[0])) if kt[0] else float(np.mean(roll_ms))
    achieved = P * Q * H * flop_step / (k_ms * 1e-3) / 1e12
    if ctx.prec == vl.PREC_BF16 and "tc" in ctx.voila_last_rollout_kernel():
        long_step = ms_per_step > 500.0
        peak = peaks["bf16_sustained"] if long_step else peaks["bf16_burst"]
        roof = {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak, "traffic": None,
                "peak_kind": f"bf16 {'sustained' if long_step else 'burst'}, {peaks['src']}"}
    else:
        sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
        mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
        peak = _flops_fp32_peak_tflops(sm_count, mhz)
        roof = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak, "traffic": None,
                "peak_kind": "fp32 FFMA: SMs x 128 lanes x 2 flop x max SM clock (CUDA-core kernel)"}
    # roof["traffic"]: DRAM bytes of ONE launch (dram__bytes_read.sum + dram__bytes_write.sum) from the
    # committed `ncu --set full` capture of this kernel at THIS size (full-size CFG5); null for any other
    # size or kernel (inputs are read once, per-(q, tile) partial sums written; the horizon loop never touches HBM)
    if cfg.index == 5 and not reduced and "rollout_tc2x" in ctx.voila_last_rollout_kernel():
        roof["traffic"] = 5590784 + 26686208
        roof["traffic_from"] = "profiles/r02j_rollout_tc2x_cfg5_fullsize.md (ncu --set full, the full-size launch)"
    roof.update({"kernel": ctx.voila_last_rollout_kernel(), "kernel_ms": k_ms,
                 "flop_per_unit": flop_step, "units_per_launch": P * Q * H,
                 "share_of_step": k_ms / ms_per_step})
    # HBM-bound tail of the belief update (scan + resample/gather), algorithmic bytes per particle
    row = cfg.S * esize
    belief = {"latency_us": 1e3 * float(np.mean(bu_ms)), "back_to_back_us": bu_b2b_us,
              "propose_score_us": 1e3 * float(np.mean(kt[1])) if kt[1] else None,
              "scan_us": 1e3 * float(np.mean(kt[2])) if kt[2] else None,
              "resample_gather_us": 1e3 * float(np.mean(kt[3])) if kt[3] else None}
    belief.update(_belief_roofs(N, row, kt, synth.flops_per_belief_particle(model), peaks,
                                ctx.voila_last_belief_kernel() if ctx.prec == vl.PREC_BF16 else ""))
    if N < (1 << 17):  # belief updates of a few thousand particles are launch-latency-bound
        for k in ("resample_roofline", "scan_roofline", "propose_score_roofline"):
            if k in belief:
                belief[k]["note"] = "latency-bound at this N: report the microseconds, not the fraction"

    # SURVEY 8d / north_star also quote the nominal figures: 2250 TFLOP/s dense bf16, ~8 TB/s HBM3e
    if roof["bound"] == "tensor":
        roof["nominal_peak"] = 2250.0
        roof["frac_of_nominal"] = roof["achieved"] / 2250.0

    porpp = _porpp_leg(ctx, dev, peaks)
    extra = {}
    all_legs = ["belief_update_cfg4", "rollout_cfg3", "progressive_widening", "diffusion_teacher"]
    if args.legs is not None:
        legs = [x for x in args.legs.split(",") if x]
    else:
        legs = all_legs if (args.config == DEFAULT_CONFIG and not reduced and not args.no_legs) else []
    # BASELINE.json's metric is "rollout steps/sec AND belief-update latency": the latency half is defined
    # on config 4 (2^20 particles), the paper-shaped rollout on config 3; then the SURVEY 8(f) rows
    if "belief_update_cfg4" in legs:
        extra["belief_update_cfg4"] = _leg_belief_cfg4(vl, synth, dev, local, peaks, flush)
    if "rollout_cfg3" in legs:
        extra["rollout_cfg3"] = _leg_rollout_cfg3(vl, synth, dev, local, peaks, flush)
    if "progressive_widening" in legs:
        extra["progressive_widening"] = _leg_pw(vl, synth, dev, local, peaks, flush)
    if "diffusion_teacher" in legs:
        extra["diffusion_teacher"] = _leg_diffusion(vl, synth, dev, local, peaks)

    cpu_v, cores, desc, _ = _oracle_sample(cfg, model, inp, target_s=args.cpu_seconds)
    cpu_1t = _oracle_one_thread(cfg, model, inp)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if ctx.prec == vl.PREC_BF16 else "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "P": P, "Q": Q, "H": H, "N": N, "S": cfg.S, "O": cfg.O,
                   "A": cfg.A, "Nz": cfg.Nz, "hidden": cfg.hidden, "parallelism": "replicas only",
                   "l2": "flushed between timed iterations (256 MiB write)",
                   "chained_belief": chain, "reduced": reduced},
        "rollout_ms": float(np.mean(roll_ms)), "belief_update": belief,
        "roofline": roof,
        "cpu_baseline": {"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                         "value_one_thread": cpu_1t},
        "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "porpp_backup": porpp,
    }
    line.update(extra)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="voila", choices=["voila", "reference"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "ffma", "tcgen05"])
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--legs", default=None,
                    help="comma list of the extra legs to run whatever the config (profiling runs): "
                         "belief_update_cfg4,rollout_cfg3,progressive_widening,diffusion_teacher")
    ap.add_argument("--no-legs", action="store_true",
                    help="skip the config-4 belief-update and config-3 rollout legs of the default line")
    # size overrides for profiling runs (ncu replays every launch ~40 times); the line then says
    # "reduced": true in config and is not a bench value
    for name in ("P", "Q", "H", "N"):
        ap.add_argument(f"--{name}", type=int, default=0)
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "voila":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_voila(args)


if __name__ == "__main__":
    main()
