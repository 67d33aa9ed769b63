"""-m gpu: the work order of the fused walk (split_group, paper_1406_6158_b200/csrc/common.cuh).  With few sink groups
per resident warp the longest groups of the previous fused walk are handed out first, the heaviest cut into 2 or 4
sink ranges.  The lists are the groups' lists whatever the order (T12-T13): list lengths and pair counts stay bit-exact
against the oracle, the accelerations stay within the parity tolerance and differ from an uncut walk in the last bits
only."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from workloads import CONFIGS, make_ic

pytestmark = pytest.mark.gpu

from gpu_util import check_forces, compare_lists, make_hyb  # noqa: E402


@pytest.mark.parametrize("kind,n", [("plummer", 30011), ("hernquist", 8192)])
def test_second_fused_walk_is_cut_and_still_matches_the_oracle(kind, n):
    cfg = CONFIGS[1].with_(n=n, kind=kind)
    pos, vel = make_ic(kind, n, 5)
    h = make_hyb(cfg, pos, vel)
    h.build_tree(); h.soft_force(); h.sync()
    assert int(h.export("counts")[7]) == 0                 # no estimate yet: the ordinary sequence
    first = h.a_soft.clone(), h.a_hard.clone()
    lists = [h.export(k).copy() for k in ("ncell", "npart", "nhard")]
    inter = h.export("interactions")
    store = h.pos_m.cpu().numpy()
    h.build_tree(); h.soft_force(); h.sync()               # same positions, same tree; the work order is prepared now
    queued = int(h.export("counts")[7])
    assert queued > 0
    for a, k in zip(lists, ("ncell", "npart", "nhard")):
        assert np.array_equal(a, h.export(k))
    assert np.array_equal(inter, h.export("interactions"))
    for a, b in zip(first, (h.a_soft, h.a_hard)):
        assert not torch.equal(a, b)                       # some group was cut: its partial sums combine differently ...
        assert float((a - b).norm() / a.norm()) < 1e-6     # ... in the last bits
    t = O.Tree(store, O.params_from(cfg))
    compare_lists(h, t, O.MODE_HYBRID)
    h.build_tree(); h.sync()
    print(queued, check_forces(h, t))                      # third fused walk (cut as well) and a hard walk against the oracle
    h.close()


def test_large_runs_keep_the_morton_order():
    cfg = CONFIGS[2].with_(n=400009)
    pos, vel = make_ic(cfg.kind, cfg.n, 5)
    h = make_hyb(cfg, pos, vel)
    h.build_tree(); h.soft_force(); h.sync()
    first = h.a_soft.clone(), h.a_hard.clone()
    h.build_tree(); h.soft_force(); h.sync()
    assert int(h.export("counts")[7]) == 0
    assert torch.equal(first[0], h.a_soft) and torch.equal(first[1], h.a_hard)
    h.close()
