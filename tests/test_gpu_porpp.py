"""GPU parity: voila_porpp_backup_level (through the C ABI) against the CPU oracle of Eq. 1
(PAPER.md:46-53), element by element on seeded synthetic trees.  Run on the B200: pytest -m gpu."""
import numpy as np
import pytest

from oracle import porpp_oracle as po
from paper_2606_19729_b200 import synth, synth_tree
from tests.parity_util import TOL_FP32, t2n

pytestmark = pytest.mark.gpu


def _to_dev(torch, levels, leaves):
    dl = []
    for lv in levels:
        dl.append({k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in lv.items()})
        dl[-1]["child_off"] = dl[-1]["child_off"].to(torch.int32)
        dl[-1]["child_idx"] = dl[-1]["child_idx"].to(torch.int32)
    return dl, torch.from_numpy(leaves).cuda()


@pytest.mark.parametrize("seed,depth,A,branches,roots,eta", [
    (0, 1, 1, 0, 1, 1.0),          # one belief node, one action, no branches
    (1, 3, 4, 3, 2, 2.5),
    (2, 4, 9, 2, 5, 0.5),          # FloorPositioning-like |A| = 9
    (3, 3, 40, 2, 3, 8.0),         # more actions than lanes
    (4, 6, 6, 3, 1, 30.0),         # deep: ~10^5 leaves; sharp eta
])
def test_porpp_backup_matches_oracle(oracle, seed, depth, A, branches, roots, eta):
    import torch
    import paper_2606_19729_b200 as vl
    assert torch.cuda.is_available()
    levels, leaves = synth_tree.make_tree(seed, depth, A, branches, roots)
    V_ref, Psi_ref = po.porpp_backup(levels, leaves, eta, 0.95)
    ctx = vl.Voila(synth.make_model(synth.CONFIGS[1]))
    dl, dleaves = _to_dev(torch, levels, leaves)
    # the whole tree in ONE C-ABI call (with the root action), and level by level: same numbers
    V, Psi, root = ctx.voila_porpp_backup(dl, dleaves, eta, 0.95)
    V2, Psi2, _ = ctx.voila_porpp_backup(dl, dleaves, eta, 0.95, per_level_calls=True)
    torch.cuda.synchronize()
    for d in range(depth):
        scale = max(1.0, float(np.max(np.abs(V_ref[d]))))
        assert np.max(np.abs(t2n(V[d]) - V_ref[d])) <= TOL_FP32 * scale, f"V level {d}"
        assert np.max(np.abs(t2n(Psi[d]) - Psi_ref[d])) <= TOL_FP32 * scale, f"Psi level {d}"
        assert torch.equal(V[d], V2[d]) and torch.equal(Psi[d], Psi2[d])
    # root action: the argmax of the GPU's own root preferences (an integer decided in fp32, ties -> lowest
    # a), and the oracle's action wherever its two best preferences are further apart than the tolerance
    psi0 = t2n(Psi[0])
    assert np.array_equal(root.cpu().numpy(), po.root_action(psi0))
    ref_root = po.root_action(Psi_ref[0])
    srt = np.sort(Psi_ref[0], axis=1)
    clear = (srt[:, -1] - srt[:, -2] > 1e-3 * max(1.0, float(np.abs(Psi_ref[0]).max()))) if A > 1 else np.ones(roots, bool)
    assert np.array_equal(root.cpu().numpy()[clear], ref_root[clear])
    ctx.close()


def test_porpp_backup_argument_errors():
    import torch
    import paper_2606_19729_b200 as vl
    levels, leaves = synth_tree.make_tree(1, 2, 3, 2, 1)
    ctx = vl.Voila(synth.make_model(synth.CONFIGS[1]))
    dl, dleaves = _to_dev(torch, levels, leaves)
    for eta, gamma in [(0.0, 0.9), (-1.0, 0.9), (1.0, -0.1)]:
        with pytest.raises(vl.VoilaError):
            ctx.voila_porpp_backup(dl, dleaves, eta, gamma)
    ctx.close()
