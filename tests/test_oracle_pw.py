"""Pins for the oracle's vectorised progressive widening with batched likelihood (vo_pw_update;
PAPER.md:147-149; readings R26-R29).  CPU only.  Expected values: the plain
belief update (separately pinned) in the cases that reduce to it, an exact-integer evaluation of the
widening criterion, the KAT-pinned Philox words, and the resampler's count invariants per child belief."""
from fractions import Fraction

import numpy as np

from paper_2606_19729_b200 import synth


def _setup(cfg_idx=1, N=96, G=4, M_max=6, seed=5, equal_groups=False, lik_action_cond=0):
    cfg = synth.CONFIGS[cfg_idx]
    model = synth.make_model(cfg, lik_action_cond=lik_action_cond)
    rng = np.random.default_rng(seed)
    parts = rng.standard_normal((N, cfg.S)).astype(np.float32)
    if equal_groups:
        cuts = np.linspace(0, N, G + 1).astype(np.int32)
    else:
        cuts = np.concatenate([[0], np.sort(rng.choice(np.arange(1, N), G - 1, replace=False)), [N]]).astype(np.int32)
    acts = rng.integers(0, cfg.A, G).astype(np.int32)
    return cfg, model, rng, parts, cuts, acts


def test_single_stored_branch_is_the_belief_update(oracle):
    """One action node with one stored observation and no room to widen: every simulation attaches to
    it, and the call IS the SIR update with that observation, bit for bit."""
    cfg, model, rng, parts, _, _ = _setup(N=200)
    om = oracle.OracleModel(model)
    o = rng.standard_normal(cfg.O).astype(np.float32)
    w = rng.uniform(0.1, 1.0, 200).astype(np.float32)
    for a in (0, 3):
        ref = om.belief_update(parts, a, o, w, seed=99)
        out = om.pw_update(parts, [0, 200], [a], [17], [1], o.reshape(1, 1, -1), 0.7, 0.4, w, seed=99)
        for k in ("proposals", "logits", "post_weights", "ancestors", "particles"):
            assert np.array_equal(out[k], ref[k]), k
        assert np.all(out["sim_branch"] == 0) and np.all(out["opened"] == 0)
        assert out["visit_count"][0] == 217 and out["branch_count"][0] == 1
        np.testing.assert_allclose(out["weights"], 1.0 / 200)


def test_identical_branch_observations_give_identical_scores(oracle):
    """M stored branches holding the SAME observation: the score of a successor state does not depend on
    the branch it was attached to, and equals the belief update's logit for that observation."""
    cfg, model, rng, parts, _, _ = _setup(N=150)
    om = oracle.OracleModel(model)
    o = rng.standard_normal(cfg.O).astype(np.float32)
    M = 5
    ref = om.belief_update(parts, 2, o, None, seed=7)
    out = om.pw_update(parts, [0, 150], [2], [10 ** 6], [M], np.tile(o, (1, M, 1)), 1.0, 0.5, None, seed=7)
    assert np.array_equal(out["logits"], ref["logits"])
    assert set(np.unique(out["sim_branch"])) == set(range(M)) and np.all(out["opened"] == 0)


def _exact_widening(n0, c0, n_new, k_num, k_den, M_max):
    """alpha = 1/2, k = k_num/k_den: C < k sqrt(n)  <=>  C^2 k_den^2 < k_num^2 n  (exact integers).
    Returns the branch count after each of the n_new visits and which visits opened a branch."""
    C, opened, counts = c0, [], []
    for j in range(n_new):
        n = n0 + j + 1
        grow = C < M_max and Fraction(C * C * k_den * k_den) < Fraction(k_num * k_num * n)
        opened.append(int(grow))
        C += int(grow)
        counts.append(C)
    return counts, opened


def test_widening_counts_exact_arithmetic(oracle):
    """The criterion |C(a)| < k_o N(a)^alpha_o visit by visit against an exact-integer
    evaluation (alpha = 1/2, rational k), including the visits where k sqrt(n) is an exact integer."""
    cfg, model, rng, parts, _, _ = _setup(N=400)
    om = oracle.OracleModel(model)
    for (k_num, k_den, n0, c0, M_max) in [(1, 1, 0, 0, 64), (2, 1, 0, 0, 64), (3, 2, 5, 1, 64), (1, 2, 0, 0, 64),
                                           (2, 1, 0, 0, 7), (1, 1, 100, 3, 64)]:
        bo = np.zeros((1, M_max, cfg.O), np.float32)
        bo[0, :c0] = rng.standard_normal((c0, cfg.O))
        out = om.pw_update(parts, [0, 400], [1], [n0], [c0], bo, k_num / k_den, 0.5, None, seed=3)
        counts, opened = _exact_widening(n0, c0, 400, k_num, k_den, M_max)
        assert out["opened"].tolist() == opened, (k_num, k_den, n0, c0)
        assert out["branch_count"][0] == counts[-1] and out["visit_count"][0] == n0 + 400
        # once the count has caught up with the threshold it IS ceil(k sqrt(n)) (capped), SURVEY f1 pin
        n = n0 + 400
        if counts[-1] < M_max and counts[-1] > c0:
            c = counts[-1]
            assert (c - 1) ** 2 * k_den ** 2 < k_num ** 2 * n <= c ** 2 * k_den ** 2
        # a simulation that opens a branch is attached to it; the others to an existing branch picked by
        # their Philox word (stream 6, counter (i, 0, 0)): b = (x * C) >> 32
        C = c0
        for i in range(400):
            if opened[i]:
                assert out["sim_branch"][i] == C
                C += 1
            else:
                x = oracle.philox4x32_10([i, 0, 0, 6 << 16], [3, 0])[0]
                assert out["sim_branch"][i] == (int(x) * C) >> 32


def test_new_branches_store_the_sampled_observation(oracle):
    """o_i = f_Z(s'_i, a, w_Z(i)) recomposed from separately pinned pieces: the proposals of
    the belief update, the stream-5 normals and the MLP forward; opened branches store exactly these rows."""
    cfg, model, rng, parts, cuts, acts = _setup(N=64, G=3, M_max=8)
    om = oracle.OracleModel(model)
    G = 3
    out = om.pw_update(parts, cuts, acts, np.zeros(G), np.zeros(G), np.zeros((G, 8, cfg.O)), 1.5, 0.6, None, seed=11)
    for g in range(G):
        ref = om.belief_update(parts, int(acts[g]), np.zeros(cfg.O, np.float32), None, seed=11)
        sl = slice(cuts[g], cuts[g + 1])
        assert np.array_equal(out["proposals"][sl], ref["proposals"][sl])
        for i in range(cuts[g], cuts[g + 1]):
            x = np.concatenate([out["proposals"][i], np.eye(cfg.A, dtype=np.float32)[acts[g]],
                                oracle.normals(11, i, 0, 0, 5, cfg.Nz)])
            np.testing.assert_allclose(out["obs"][i], om.mlp_forward(1, x[None])[0], rtol=1e-6, atol=1e-7)
            if out["opened"][i]:
                assert np.array_equal(out["branch_obs"][g, out["sim_branch"][i]], out["obs"][i])
        assert out["opened"][cuts[g]] == 1  # the first visit of an empty action node always widens


def test_child_beliefs_resample_among_their_members(oracle):
    """Every (action node, branch) pair that received simulations is resampled by itself: ancestors stay
    inside the child, are non-decreasing along its members, their counts are floor/ceil of n*wbar, and
    equal the stage-level resampler run on the child's own weights with the child's offset word."""
    cfg, model, rng, parts, cuts, acts = _setup(N=600, G=5, M_max=6, seed=8)
    om = oracle.OracleModel(model)
    G, M_max = 5, 6
    w = rng.uniform(0.05, 1.0, 600).astype(np.float32)
    bc0 = np.array([0, 2, 6, 1, 3])
    bo = rng.standard_normal((G, M_max, cfg.O)).astype(np.float32)
    out = om.pw_update(parts, cuts, acts, [0, 9, 50, 3, 20], bc0, bo, 1.2, 0.55, w, seed=21)
    seen = 0
    for g in range(G):
        idx = np.arange(cuts[g], cuts[g + 1])
        for b in range(out["branch_count"][g]):
            mem = idx[out["sim_branch"][idx] == b]
            if mem.size == 0:
                continue
            seen += 1
            anc = out["ancestors"][mem]
            assert np.all(np.isin(anc, mem)) and np.all(np.diff(anc) >= 0)
            v = out["post_weights"][mem]
            assert v.max() == 1.0
            wbar, st = oracle.normalised_weights(v)
            cnt = np.array([(anc == i).sum() for i in mem])
            assert st == 0 and cnt.sum() == mem.size
            assert np.all(cnt >= np.floor(mem.size * wbar - 1e-9)) and np.all(cnt <= np.ceil(mem.size * wbar + 1e-9))
            x0 = oracle.philox4x32_10([g * M_max + b, 0, 0, 4 << 16], [21, 0])[0]
            a_loc, st = oracle.resample_systematic_x0(v, int(x0))
            assert st == 0 and np.array_equal(anc, mem[a_loc])
            assert np.array_equal(out["particles"][mem], out["proposals"][anc])
            np.testing.assert_allclose(out["weights"][mem], 1.0 / mem.size)
    assert seen >= 10 and np.all(out["seg_status"] == 0)


def test_zero_weight_child_keeps_its_members(oracle):
    cfg, model, rng, parts, _, _ = _setup(N=40)
    om = oracle.OracleModel(model)
    bo = rng.standard_normal((1, 2, cfg.O)).astype(np.float32)
    first = om.pw_update(parts, [0, 40], [0], [10 ** 6], [2], bo, 1.0, 0.5, None, seed=2)
    w = np.where(first["sim_branch"] == 1, 0.0, 1.0).astype(np.float32)
    out = om.pw_update(parts, [0, 40], [0], [10 ** 6], [2], bo, 1.0, 0.5, w, seed=2)
    assert out["seg_status"].tolist() == [0, 1]
    dead = np.flatnonzero(first["sim_branch"] == 1)
    assert np.array_equal(out["ancestors"][dead], dead)
    assert np.array_equal(out["particles"][dead], out["proposals"][dead])
