"""-m gpu: the sink-sharded evaluation on one GPU (hyb_set_sink_range, hyb_kick_drift, sharded.ShardedHyb).
One GPU is all the pool offers, so the ranks are emulated one after the other (no kernel waits on another):
the sum over complementary sink ranges is the full result (bit for bit while no group is cut into sink ranges, to
the last bits otherwise), and the call-by-call cycle equals hyb_step bit for bit."""
import numpy as np
import pytest
import torch

from workloads import CONFIGS, make_ic

pytestmark = pytest.mark.gpu

from gpu_util import make_hyb  # noqa: E402


def test_ranges_sum_to_the_full_result():
    cfg = CONFIGS[2].with_(n=200003)
    pos, vel = make_ic(cfg.kind, cfg.n, 3)
    h = make_hyb(cfg, pos, vel)
    h.build_tree(); h.soft_force(); h.sync()
    full_s, full_h = h.a_soft.clone(), h.a_hard.clone()
    want = h.export("interactions")
    h.hard_force(); h.sync()
    full_h2 = h.a_hard.clone()
    h.export("interactions")
    from paper_1406_6158_b200.sharded import sink_ranges
    for world in (2, 3):
        b = sink_ranges(cfg.n, world)
        sum_s, sum_h, sum_h2 = torch.zeros_like(full_s), torch.zeros_like(full_h), torch.zeros_like(full_h)
        got = np.zeros(4, np.uint64)
        for r in range(world):
            h.set_sink_range(b[r], b[r + 1])
            h.soft_force(); h.sync()
            nz = (h.a_soft.abs().sum(dim=1) > 0).nonzero().flatten()
            assert nz.numel() > 0
            sum_s += h.a_soft; sum_h += h.a_hard
            got += h.export("interactions")
            h.hard_force(); h.sync()
            sum_h2 += h.a_hard
            h.export("interactions")
        # (a repeated walk may cut its longest groups into sink ranges, whose partial sums combine in another order)
        assert float((sum_s - full_s).norm() / full_s.norm()) < 1e-6 and float((sum_h - full_h).norm() / full_h.norm()) < 1e-6
        assert np.array_equal(got[:3], want[:3])                         # every pair evaluated by exactly one rank
        # hard-only walk: heavy groups are cut into sink ranges whose partial sums combine in another order
        assert float((sum_h2 - full_h2).norm() / full_h2.norm()) < 1e-6
    h2 = make_hyb(CONFIGS[2].with_(n=400009), *make_ic(cfg.kind, 400009, 3))       # above the size where the fused walk follows a work order
    h2.build_tree(); h2.soft_force(); h2.sync()
    full = h2.a_soft.clone(), h2.a_hard.clone()
    b = sink_ranges(400009, 2)
    acc = [torch.zeros_like(full[0]), torch.zeros_like(full[1])]
    for r in range(2):
        h2.set_sink_range(b[r], b[r + 1])
        h2.soft_force(); h2.sync()
        acc[0] += h2.a_soft; acc[1] += h2.a_hard
    assert torch.equal(acc[0], full[0]) and torch.equal(acc[1], full[1])     # Morton order, no group cut: the same bits
    h2.close()
    from paper_1406_6158_b200 import HybError
    with pytest.raises(HybError):
        h.step(1)                                                        # a partial range needs the caller's exchange
    h.set_sink_range(0, cfg.n)
    h.close()


@pytest.mark.parametrize("split,n_sub", [(1, 4), (0, 4), (1, 3), (1, 1)])
def test_call_by_call_cycle_equals_hyb_step(split, n_sub):
    """(n_sub = 3, 1: an odd number of builds per hyb_step call -- inside the call the builds move the store between the
    caller's arrays and the workspace copy, and it has to be home again when the call returns)"""
    from types import SimpleNamespace
    from paper_1406_6158_b200.sharded import ShardedHyb
    cfg = CONFIGS[1].with_(n=50021, split=split, n_sub=n_sub)
    pos, vel = make_ic(cfg.kind, cfg.n, 8)
    ref = make_hyb(cfg, pos, vel)
    ref.step(1); ref.step(1); ref.sync()                   # (two calls: n_sub builds in the second one)
    h = make_hyb(cfg, pos, vel)
    sh = ShardedHyb(h, SimpleNamespace(split=cfg.split, n_sub=cfg.n_sub, dt_soft=cfg.dt_soft), 0, 1, lambda t: None)
    sh.step(2); h.sync()
    for a, b in ((h.pos_m, ref.pos_m), (h.vel, ref.vel), (h.a_soft, ref.a_soft), (h.a_hard, ref.a_hard), (h.ids, ref.ids)):
        assert torch.equal(a, b)
    h.close(); ref.close()
