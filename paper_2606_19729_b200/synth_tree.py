"""Seeded synthetic belief trees for the PORPP preference backup (no method arithmetic: numpy draws
and index bookkeeping only; serves both the oracle and the CUDA path).

Level d: `nb` belief nodes x A action nodes; action node j = b * A + a owns 0..max_branches
observation branches (belief nodes of level d + 1, numbered in creation order) with weights
Z(b,a,o) that sum to 1 over the branches (Monte-Carlo frequencies)."""
import numpy as np


def make_tree(seed, depth, n_actions, max_branches, root_beliefs=1):
    rng = np.random.default_rng(seed)
    levels = []
    nb = root_beliefs
    for _ in range(depth):
        na = nb * n_actions
        counts = rng.integers(0, max_branches + 1, size=na)
        off = np.zeros(na + 1, np.int32)
        off[1:] = np.cumsum(counts)
        nnz = int(off[-1])
        w = rng.uniform(0.1, 1.0, size=nnz).astype(np.float32)
        for j in range(na):
            s = slice(off[j], off[j + 1])
            if off[j + 1] > off[j]:
                w[s] /= w[s].sum()
        logits = rng.standard_normal((nb, n_actions))
        logpi0 = (logits - np.log(np.exp(logits).sum(axis=1, keepdims=True))).astype(np.float32)
        levels.append(dict(R=rng.standard_normal((nb, n_actions)).astype(np.float32), logpi0=logpi0,
                           child_off=off, child_idx=np.arange(nnz, dtype=np.int32), child_w=w))
        nb = nnz
    leaves = rng.standard_normal(nb).astype(np.float32)
    return levels, leaves
