"""Pins for the oracle's terminal regions (R25).
CPU only.  Expected values: closed forms (truncated geometric series), an independent numpy
simulation of a FloorPositioning-shaped grid world, bit equality with the plain rollout when no
region is ever reached."""
import numpy as np

from paper_2606_19729_b200 import synth
from paper_2606_19729_b200.synth import (ACT_NONE, MLPSpec, ModelSpec, R_LINEAR, TerminalSpec)


def _towers(rng, S, O):
    return (synth.make_mlp(rng, [O, 4, 3], ACT_NONE), synth.make_mlp(rng, [S, 4, 3], ACT_NONE))


def _walk_model(rng, S, O, A, Nz, gamma, moves, c0, cost, terminal):
    """Deterministic walk s' = s + moves[a] (f_T = [I | moves^T | 0]), constant reward c0 + cost[a]."""
    gin = S + A + Nz
    WT = np.zeros((S, gin), np.float32)
    WT[:, :S] = np.eye(S)
    WT[:, S:S + A] = moves.T
    f_T = MLPSpec([gin, S], ACT_NONE, [WT], [np.zeros(S, np.float32)])
    f_Z = synth.make_mlp(rng, [gin, O], ACT_NONE)
    lo, ls = _towers(rng, S, O)
    c = np.zeros(S + 1, np.float32)
    c[-1] = c0
    return ModelSpec(S, O, A, Nz, f_T, f_Z, lo, ls, gamma=gamma, reward_kind=R_LINEAR, reward_param=c,
                     action_cost=cost, terminal=terminal)


def test_truncated_geometric_series(oracle):
    """1-D walk to the right by 0.25 per step from s0 = 0, goal ball |s - 2| <= 0.1 (terminates, +100),
    reward -1 per step: the state enters at t* = 8, so G = -(1 - g^8)/(1 - g) + g^8 * 100, the state
    freezes at 2.0 and later steps add nothing (H = 8, 9, 20 give the same G; H <= 8 never arrives)."""
    rng = np.random.default_rng(11)
    gamma = 0.9
    term = TerminalSpec([np.array([2.0], np.float32)], np.array([0.1], np.float32),
                        np.array([100.0], np.float32), np.array([1], np.int32))
    m = _walk_model(rng, 1, 2, 2, 1, gamma, np.array([[0.25], [-0.25]], np.float32), -1.0, None, term)
    om = oracle.OracleModel(m)
    s0 = np.zeros((1, 1), np.float32)
    for H in (5, 8, 9, 20):
        seqs = np.zeros((1, H), np.int32)
        out = om.rollout_values_term(s0, seqs, None, seed=3)
        if H <= 8:
            expect = -(1 - gamma ** H) / (1 - gamma)
            assert out["t_term"][0, 0] == H
            np.testing.assert_allclose(out["final_states"][0, 0, 0], 0.25 * H, rtol=1e-6)
        else:
            expect = -(1 - gamma ** 8) / (1 - gamma) + gamma ** 8 * 100.0
            assert out["t_term"][0, 0] == 8
            np.testing.assert_allclose(out["final_states"][0, 0, 0], 2.0, rtol=1e-6)
        np.testing.assert_allclose(out["returns"][0, 0], expect, rtol=1e-5)
        np.testing.assert_allclose(out["values"][0], expect, rtol=1e-5)
        G, states, obs = om.rollout_trajectory(s0[0], seqs[0], 0, 0, 3)
        np.testing.assert_allclose(G, expect, rtol=1e-5)
        if H > 8:
            assert np.all(states[8:] == states[8]) and np.all(obs[8:] == 0.0) and np.any(obs[7] != 0.0)


def test_everything_terminal_at_step_zero(oracle):
    """A stopping ball that contains every particle: G = reward_k exactly, the particles come back
    unchanged, the witness is zero (no step was taken), whatever the step reward is."""
    rng = np.random.default_rng(12)
    cfg = synth.CONFIGS[1]
    term = TerminalSpec([np.zeros(2, np.float32)], np.array([1e3], np.float32), np.array([7.5], np.float32),
                        np.array([1], np.int32))
    m = synth.make_model(cfg, action_cost=True).replace(terminal=term)
    om = oracle.OracleModel(m)
    inp = synth.make_inputs(cfg, P=17, Q=3, H=6)
    out = om.rollout_values_term(inp.particles, inp.action_seqs, None, seed=9)
    assert np.all(out["returns"] == np.float32(7.5)) and np.all(out["t_term"] == 0)
    np.testing.assert_allclose(out["values"], 7.5, rtol=1e-6)
    assert np.all(out["witness"] == 0.0)
    assert np.array_equal(out["final_states"][1], inp.particles)


def test_unreached_regions_change_nothing(oracle):
    """Regions that no trajectory enters (and no region at all) reproduce the plain rollout bit for bit."""
    cfg = synth.CONFIGS[1]
    base = synth.make_model(cfg, action_cost=True)
    far = TerminalSpec([np.array([50.0, 50.0], np.float32), np.array([-80.0], np.float32)],
                       np.array([1.0, 2.0], np.float32), np.array([100.0, -100.0], np.float32),
                       np.array([1, 0], np.int32))
    inp = synth.make_inputs(cfg, P=40, Q=5, H=10)
    V0, W0, G0 = oracle.OracleModel(base).rollout_values(inp.particles, inp.action_seqs, None, 4, want_returns=True)
    out = oracle.OracleModel(base.replace(terminal=far)).rollout_values_term(inp.particles, inp.action_seqs, None, 4)
    assert np.array_equal(out["values"], V0) and np.array_equal(out["witness"], W0)
    assert np.array_equal(out["returns"], G0) and np.all(out["t_term"] == 10)
    assert np.all(out["margin"] > 40.0)


def test_floor_positioning_shaped_grid_world(oracle):
    """eight compass moves of 0.05 and STAY, +100 at the correct goal (terminates), -100 at
    the incorrect goal (does not terminate), -1 per non-terminal action, gamma = 0.99.  The oracle against
    an independent numpy simulation of exactly that, on random starts and random action sequences."""
    rng = np.random.default_rng(13)
    d = 0.05
    moves = np.array([[d, 0], [d, d], [0, d], [-d, d], [-d, 0], [-d, -d], [0, -d], [d, -d], [0, 0]], np.float32)
    A, H, P, Q, gamma = 9, 40, 64, 12, 0.99
    good, bad = np.array([0.3, 0.2], np.float32), np.array([-0.25, 0.1], np.float32)
    term = TerminalSpec([good, bad], np.array([0.12, 0.12], np.float32), np.array([100.0, -100.0], np.float32),
                        np.array([1, 0], np.int32))
    cost = np.full(A, -1.0, np.float32)
    m = _walk_model(rng, 2, 4, A, 2, gamma, moves, 0.0, cost, term)
    om = oracle.OracleModel(m)
    starts = rng.uniform(-0.5, 0.5, (P, 2)).astype(np.float32)
    seqs = rng.integers(0, A, (Q, H), dtype=np.int32)
    w = rng.uniform(0.2, 1.0, P).astype(np.float32)
    out = om.rollout_values_term(starts, seqs, w, seed=21)
    Gref = np.zeros((Q, P))
    tref = np.full((Q, P), H)
    sref = np.zeros((Q, P, 2))
    near = np.zeros((Q, P), bool)
    for q in range(Q):
        for p in range(P):
            s = starts[p].astype(np.float64)
            for t in range(H):
                dg, db = np.linalg.norm(s - good), np.linalg.norm(s - bad)
                near[q, p] |= abs(dg - 0.12) < 1e-4 or abs(db - 0.12) < 1e-4
                if dg <= 0.12:
                    Gref[q, p] += gamma ** t * 100.0
                    tref[q, p] = t
                    break
                Gref[q, p] += gamma ** t * ((-100.0 if db <= 0.12 else 0.0) - 1.0)
                s = s + moves[seqs[q, t]].astype(np.float64)
            sref[q, p] = s
    ok = ~near  # membership decisions closer than 1e-4 to the boundary may differ between fp32 and fp64
    assert ok.mean() > 0.97 and (tref < H).mean() > 0.05 and (Gref < -150).mean() > 0.05
    assert np.array_equal(out["t_term"][ok], tref[ok])
    np.testing.assert_allclose(out["returns"][ok], Gref[ok], rtol=2e-5, atol=2e-4)
    np.testing.assert_allclose(out["final_states"][ok], sref[ok], atol=2e-5)
    assert np.all(out["margin"][ok] >= 1e-4 * 0.5)
    if ok.all():
        wbar = w.astype(np.float64) / w.astype(np.float64).sum()
        np.testing.assert_allclose(out["values"], Gref @ wbar, rtol=2e-5, atol=2e-4)


def test_witness_stops_at_termination(oracle):
    """The observation witness sums gamma^t o_{t+1} over the steps actually taken: for a trajectory that
    terminates at t*, it equals the witness of the same rollout cut at H = t*."""
    rng = np.random.default_rng(14)
    term = TerminalSpec([np.array([1.0], np.float32)], np.array([0.05], np.float32), np.array([10.0], np.float32),
                        np.array([1], np.int32))
    m = _walk_model(rng, 1, 3, 2, 2, 0.95, np.array([[0.25], [-0.25]], np.float32), -1.0, None, term)
    om = oracle.OracleModel(m)
    s0 = np.zeros((1, 1), np.float32)
    seqs = np.zeros((1, 12), np.int32)
    full = om.rollout_values_term(s0, seqs, None, seed=6)
    assert full["t_term"][0, 0] == 4
    cut = oracle.OracleModel(m.replace(terminal=None)).rollout_values_term(s0, seqs[:, :4], None, seed=6)
    np.testing.assert_allclose(full["witness"], cut["witness"], rtol=1e-6, atol=1e-7)
    assert np.any(full["witness"] != 0.0)
