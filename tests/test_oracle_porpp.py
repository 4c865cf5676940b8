"""Pins for the oracle of the PORPP preference backup (Eq. 1).  CPU only."""
import numpy as np
import scipy.special

from paper_2606_19729_b200 import synth_tree
from oracle import porpp_oracle as po


def _recursive(node, eta, gamma):
    """Eq. 1 written as a recursion on a nested Python tree: node = list over actions of
    (logpi0, R, [(z, child_node), ...]); a leaf is a float."""
    if not isinstance(node, list):
        return float(node)
    psi = []
    for lp, r, branches in node:
        fut = sum(z * _recursive(ch, eta, gamma) for z, ch in branches)
        psi.append(lp / eta + r + gamma * fut)
    return scipy.special.logsumexp(eta * np.array(psi)) / eta


def _nested(levels, leaf_values, d, b):
    if d == len(levels):
        return float(leaf_values[b])
    lv = levels[d]
    A = lv["R"].shape[1]
    node = []
    for a in range(A):
        j = b * A + a
        br = [(float(lv["child_w"][c]), _nested(levels, leaf_values, d + 1, int(lv["child_idx"][c])))
              for c in range(lv["child_off"][j], lv["child_off"][j + 1])]
        node.append((float(lv["logpi0"][b, a]), float(lv["R"][b, a]), br))
    return node


def test_matches_recursive_evaluation_of_eq1():
    for seed in range(4):
        levels, leaves = synth_tree.make_tree(seed, depth=3, n_actions=3, max_branches=3, root_beliefs=2)
        V, Psi = po.porpp_backup(levels, leaves, eta=2.5, gamma=0.9)
        for b in range(levels[0]["R"].shape[0]):
            ref = _recursive(_nested(levels, leaves, 0, b), 2.5, 0.9)
            assert abs(V[0][b] - ref) < 1e-10 * max(1.0, abs(ref))


def test_regular_tree_geometric_series():
    """Uniform reference policy, constant reward r, one branch per action, leaves 0:
    V_d = r + gamma V_{d+1}  ->  V_0 = r (1 - gamma^D) / (1 - gamma), whatever eta and A."""
    r, gamma, D, A = 0.7, 0.95, 6, 4
    levels = []
    nb = 1
    for d in range(D):
        na = nb * A
        levels.append(dict(R=np.full((nb, A), r), logpi0=np.full((nb, A), -np.log(A)),
                           child_off=np.arange(na + 1), child_idx=np.arange(na), child_w=np.ones(na)))
        nb = na
    for eta in (0.3, 1.0, 20.0):
        V, _ = po.porpp_backup(levels, np.zeros(nb), eta, gamma)
        assert abs(V[0][0] - r * (1 - gamma ** D) / (1 - gamma)) < 1e-9


def test_large_eta_is_the_max_backup():
    levels, leaves = synth_tree.make_tree(7, depth=3, n_actions=4, max_branches=2, root_beliefs=1)
    eta = 1e4
    V, Psi = po.porpp_backup(levels, leaves, eta, 0.9)
    # hard max backup (value iteration on the tree); the prior term vanishes as 1/eta
    v_next = np.asarray(leaves, np.float64)
    for d in range(len(levels) - 1, -1, -1):
        lv = levels[d]
        nb, A = lv["R"].shape
        q = np.zeros((nb, A))
        for j in range(nb * A):
            s = slice(lv["child_off"][j], lv["child_off"][j + 1])
            q[j // A, j % A] = lv["R"][j // A, j % A] + 0.9 * np.dot(lv["child_w"][s], v_next[lv["child_idx"][s]])
        v_next = q.max(axis=1)
    assert abs(V[0][0] - v_next[0]) < 5e-3


def test_lse_against_scipy_and_shift_invariance():
    rng = np.random.default_rng(0)
    psi = rng.standard_normal(9) * 5
    for eta in (0.1, 1.0, 7.0):
        ref = scipy.special.logsumexp(eta * psi) / eta
        assert abs(po.log_sum_exp_eta(psi, eta) - ref) < 1e-12 * max(1, abs(ref))
        assert abs(po.log_sum_exp_eta(psi + 3.25, eta) - (ref + 3.25)) < 1e-10
    assert abs(po.log_sum_exp_eta(np.array([800.0, 800.0]), 2.0) - (800.0 + np.log(2) / 2)) < 1e-9  # no overflow


def test_single_action_and_no_children():
    levels = [dict(R=np.array([[1.5]]), logpi0=np.array([[0.0]]), child_off=np.array([0, 0]),
                   child_idx=np.zeros(0, np.int32), child_w=np.zeros(0))]
    V, Psi = po.porpp_backup(levels, np.zeros(0), 3.0, 0.9)
    assert V[0][0] == 1.5 and Psi[0][0, 0] == 1.5


def test_root_action_is_the_greedy_action_of_the_max_backup():
    """eta -> infinity: argmax_a Psi(b0, a) is the greedy action of value iteration on the tree (computed
    independently here with numpy); for finite eta it is numpy's argmax of the root preferences, ties -> lowest a."""
    for seed in (3, 5, 9):
        levels, leaves = synth_tree.make_tree(seed, depth=3, n_actions=5, max_branches=3, root_beliefs=4)
        V, Psi = po.porpp_backup(levels, leaves, 1e4, 0.9)
        v_next = np.asarray(leaves, np.float64)
        for d in range(len(levels) - 1, -1, -1):
            lv = levels[d]
            nb, A = lv["R"].shape
            q = np.zeros((nb, A))
            for j in range(nb * A):
                s = slice(lv["child_off"][j], lv["child_off"][j + 1])
                q[j // A, j % A] = lv["R"][j // A, j % A] + 0.9 * np.dot(lv["child_w"][s], v_next[lv["child_idx"][s]])
            v_next = q.max(axis=1)
        srt = np.sort(q, axis=1)
        clear = srt[:, -1] - srt[:, -2] > 1e-2
        assert clear.any()
        assert np.array_equal(po.root_action(Psi[0])[clear], q.argmax(axis=1)[clear])
        _, Psi2 = po.porpp_backup(levels, leaves, 2.0, 0.9)
        assert np.array_equal(po.root_action(Psi2[0]), np.argmax(Psi2[0], axis=1))
    tie = np.array([[1.0, 3.0, 3.0, -1.0], [np.nan, 0.5, 0.5, 0.2]])
    assert po.root_action(tie).tolist() == [1, 1]
