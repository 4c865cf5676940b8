"""CPU oracle of the PORPP preference backup (Eq. 1) -- TEST INFRASTRUCTURE ONLY.

    V(b)     = (1/eta) log sum_a exp(eta Psi(b, a))                         =: [L_eta Psi](b)
    Psi(b,a) = (1/eta) log pi0(a|b) + R(b,a) + gamma sum_o Z(b,a,o) [L_eta Psi](tau(b,a,o))

on a belief tree stored the way VOPP stores it, as a collection of tensors: level d
holds `nb` belief nodes, every belief node has A action nodes (action node j = b * A + a), and an
action node owns a (possibly empty) list of observation branches = belief nodes of level d + 1,
given in CSR form with the Monte-Carlo estimates Z(b,a,o) as weights.  Belief nodes of the level
below the last action level are leaves with given values (0 for a truncated search).

Plain numpy in float64, one belief node at a time, in the order of Eq. 1; no vectorisation tricks.
Only tests/ may import this module; it shares no code with the CUDA path.
Pins (tests/test_oracle_porpp.py): a recursive evaluation of Eq. 1 on nested Python trees, the
geometric-series closed form of a regular tree with uniform reference policy, eta -> infinity
(max backup), scipy.special.logsumexp, shift invariance."""
import numpy as np


def log_sum_exp_eta(psi, eta):
    """[L_eta psi] = (1/eta) log sum_a exp(eta psi_a), max-shifted."""
    psi = np.asarray(psi, np.float64)
    m = np.max(psi)
    if not np.isfinite(m):
        return float(m)
    return float(m + np.log(np.sum(np.exp(eta * (psi - m)))) / eta)


def root_action(psi_root):
    """argmax_a Psi(b0, a) for every root belief (ties -> lowest a): the action the planner returns for
    the current belief (the preferences Psi ARE the policy's scores)."""
    psi_root = np.asarray(psi_root, np.float64)
    out = np.zeros(psi_root.shape[0], np.int32)
    for b in range(psi_root.shape[0]):
        best = -1
        for a in range(psi_root.shape[1]):  # a NaN preference never wins; all NaN -> action 0
            if psi_root[b, a] == psi_root[b, a] and (best < 0 or psi_root[b, a] > psi_root[b, best]):
                best = a
        out[b] = max(best, 0)
    return out


def porpp_backup(levels, leaf_values, eta, gamma):
    """levels[d] = dict(R [nb, A], logpi0 [nb, A], child_off [nb*A + 1], child_idx [nnz], child_w [nnz]);
    leaf_values [number of belief nodes below the last action level] (may be empty).
    Returns (V, Psi): lists over depth of [nb] and [nb, A] float64 arrays."""
    D = len(levels)
    V = [None] * D
    Psi = [None] * D
    v_next = np.asarray(leaf_values, np.float64)
    for d in range(D - 1, -1, -1):
        lv = levels[d]
        R = np.asarray(lv["R"], np.float64)
        lp = np.asarray(lv["logpi0"], np.float64)
        off, idx, w = lv["child_off"], lv["child_idx"], np.asarray(lv["child_w"], np.float64)
        nb, A = R.shape
        psi = np.zeros((nb, A))
        v = np.zeros(nb)
        for b in range(nb):
            for a in range(A):
                j = b * A + a
                future = 0.0
                for c in range(off[j], off[j + 1]):
                    future += w[c] * v_next[idx[c]]
                psi[b, a] = lp[b, a] / eta + R[b, a] + gamma * future
            v[b] = log_sum_exp_eta(psi[b], eta)
        V[d], Psi[d] = v, psi
        v_next = v
    return V, Psi
