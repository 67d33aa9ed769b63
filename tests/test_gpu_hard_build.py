"""-m gpu: the tree hyb_step builds in front of a hard-only force evaluation (hyb_build_tree_hard; PAPER.md:87,
202) against the oracle: sink groups are sibling runs of at most group_max / 2 sinks (HYB_GROUP_AUTO, R17), the
upsweep computes tight boxes only.  Everything a hard walk reads is compared bit for bit, its list lengths
too, and the hard force within rms 1e-5 / max 1e-4 -- at cfg0, at the benchmark size (every particle) and at
N = 2^24 (sampled groups).  Also: boundary behaviour the advisor asked for (build twice, recover from an error
on the same context, no device allocation after hyb_init)."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from workloads import CONFIGS, make_ic

pytestmark = pytest.mark.gpu

from gpu_util import MAX_TOL, RMS_TOL, acc_errors, compare_lists, compare_tree, make_hyb  # noqa: E402


def _hard_params(cfg, **over):
    gm = max(cfg.group_max // 2, cfg.leaf_max) if cfg.grouping == 2 else cfg.group_max
    return O.params_from(cfg, group_max=gm, **over)


def _check_hard_build(cfg, pos, vel, gsel=None, **over):
    h = make_hyb(cfg, pos, vel, **over)
    h.build_tree_hard(); h.sync()
    t = O.Tree(pos, _hard_params(cfg, **over))
    compare_tree(h, t, boxes_only=True)
    h.hard_force(); h.sync()
    compare_lists(h, t, O.MODE_HARD, gsel)
    _, a_h, inter = t.forces(O.MODE_HARD, gsel)
    a_s, a_h2, _ = t.forces(O.MODE_HYBRID, gsel)                       # |a_total| of the same tree for the error scale
    if gsel is None:
        idx = np.arange(t.n)
        assert int(h.export("interactions")[1]) == int(inter[1])
    else:
        gf, gc = t.get("gfirst"), t.get("gcount")
        idx = np.concatenate([np.arange(gf[g], gf[g] + gc[g]) for g in gsel])
    gh = h.a_hard.cpu().numpy()[:, :3]
    rms, mx = acc_errors(gh[idx], a_h[idx], (a_s + a_h2)[idx])
    assert rms < RMS_TOL and mx < MAX_TOL, (rms, mx)
    # a boxes-only tree must not serve a soft walk
    from paper_1406_6158_b200 import HybError
    with pytest.raises(HybError) as ei:
        h.soft_force()
    assert ei.value.code == -5
    h.close()
    return rms, mx


@pytest.mark.parametrize("hard_cut", [0, 1])
def test_cfg0_hard_build(hard_cut):
    cfg = CONFIGS[0]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    print(_check_hard_build(cfg, pos, vel, hard_cut=hard_cut))
    cfg = CONFIGS[1].with_(n=30011)
    pos, vel = make_ic(cfg.kind, cfg.n, 23)
    print(_check_hard_build(cfg, pos, vel, hard_cut=hard_cut))


@pytest.mark.parametrize("hard_cut", [0, 1])
def test_cfg2_hard_build_full(hard_cut):
    """the configuration bench.py times: 7 of the 8 builds of a cycle are this one"""
    cfg = CONFIGS[2]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    print(_check_hard_build(cfg, pos, vel, hard_cut=hard_cut))


def test_cfg4_hard_build_sampled():
    cfg = CONFIGS[4]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel)
    h.build_tree_hard(); h.sync()
    t = O.Tree(pos, _hard_params(cfg))
    compare_tree(h, t, boxes_only=True)
    rng = np.random.default_rng(17)
    gsel = np.sort(rng.choice(t.ng, size=8192, replace=False)).astype(np.int64)
    h.hard_force(); h.sync()
    compare_lists(h, t, O.MODE_HARD, gsel)
    sub = gsel[::8]
    a_s, a_h, _ = t.forces(O.MODE_HYBRID, sub)
    gf, gc = t.get("gfirst"), t.get("gcount")
    idx = np.concatenate([np.arange(gf[g], gf[g] + gc[g]) for g in sub])
    rms, mx = acc_errors(h.a_hard.cpu().numpy()[idx, :3], a_h[idx], (a_s + a_h)[idx])
    assert rms < RMS_TOL and mx < MAX_TOL, (rms, mx)
    h.close()


def test_build_twice_then_hard_force():
    """two builds with no walk in between (positions moved): the work queue of the hard walk must hold the
    entries of the LAST build only"""
    cfg = CONFIGS[2].with_(n=150001)
    pos, vel = make_ic(cfg.kind, cfg.n, 9)
    h = make_hyb(cfg, pos, vel)
    h.build_tree(); h.hard_force(); h.sync()                  # list lengths for the estimates
    for hard in (False, True):
        (h.build_tree_hard if hard else h.build_tree)()
        h.pos_m[:, :3] *= 1.01                               # the store is in Morton order; scale keeps it so
        (h.build_tree_hard if hard else h.build_tree)()
        h.sync()
        store = h.pos_m.cpu().numpy()
        h.hard_force(); h.sync()
        t = O.Tree(store, _hard_params(cfg) if hard else O.params_from(cfg))
        compare_lists(h, t, O.MODE_HARD)
        a_s, a_h, _ = t.forces(O.MODE_HYBRID)
        rms, mx = acc_errors(h.a_hard.cpu().numpy()[:, :3], a_h, a_s + a_h)
        assert rms < RMS_TOL and mx < MAX_TOL, (hard, rms, mx)
    h.close()


def test_error_is_reported_once_and_the_context_recovers():
    from paper_1406_6158_b200 import HybError
    cfg = CONFIGS[0].with_(n=3000)
    pos, vel = make_ic(cfg.kind, cfg.n, 5)
    h = make_hyb(cfg, pos, vel)
    good = h.pos_m.clone()
    h.pos_m[17, 1] = float("nan")
    h.build_tree()
    with pytest.raises(HybError) as ei:
        h.sync()
    assert ei.value.code == -3
    with pytest.raises(HybError) as ei:                      # nothing computed from the bad input is served
        h.hard_force()
    assert ei.value.code == -5
    h.pos_m.copy_(good)
    h.build_tree(); h.sync()                                 # same context, repaired input
    t = O.Tree(pos, O.params_from(cfg))
    compare_tree(h, t)
    h.step(1); h.sync()
    good, good_v = h.pos_m.clone(), h.vel.clone()
    h.pos_m[5, 0] = float("inf")                             # the same through hyb_step
    with pytest.raises(HybError):
        h.step(1)
    h.pos_m.copy_(good); h.vel.copy_(good_v)                 # (the failed step has kicked with garbage)
    h.step(1); h.sync()
    assert np.all(np.isfinite(h.pos_m.cpu().numpy()))
    h.close()


def test_no_device_allocation_after_init():
    """include/hyb.h: a context works inside the caller's workspace (cudaMemGetInfo before / after)"""
    from workloads.domains import virtual_domains
    cfg = CONFIGS[1].with_(n=50000, mac=1)
    pos, vel = make_ic(cfg.kind, cfg.n, 3)
    h = make_hyb(cfg, pos, vel)
    h.step(1); h.build_tree(); h.sync()                      # warm: lazily loaded modules, event pool
    boxes = virtual_domains(pos, 2, 2, 2, seed=1)
    h.let_count(boxes); h.energy()
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        h.let_count(boxes); h.energy(); h.build_tree_hard(); h.hard_force(); h.build_tree(); h.soft_force(); h.step(1)
    h.sync(); torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    h.close()


def test_run_host_continues_a_run_cycle_by_cycle():
    """hyb_run_host with the state in host memory: two calls of one cycle each (the second with acc_valid = 1)
    give the same bits as two cycles on a device-resident context"""
    from paper_1406_6158_b200 import HybParams, hyb_run_host
    cfg = CONFIGS[1].with_(n=40009)
    pos, vel = make_ic(cfg.kind, cfg.n, 31)
    h = make_hyb(cfg, pos, vel)
    h.step(2); h.sync()
    P = HybParams.from_config(cfg)
    hp, hv = pos.copy(), vel.copy()
    ids = np.arange(cfg.n, dtype=np.int32)
    a_s, a_h, it0 = hyb_run_host(P, hp, hv, ids, 1, 0)
    a_s, a_h, it1 = hyb_run_host(P, hp, hv, ids, 1, 0, a_s, a_h, acc_valid=True)
    assert np.array_equal(hp, h.pos_m.cpu().numpy()) and np.array_equal(hv, h.vel.cpu().numpy())
    assert np.array_equal(ids, h.ids.cpu().numpy())
    assert np.array_equal(a_s, h.a_soft.cpu().numpy()) and np.array_equal(a_h, h.a_hard.cpu().numpy())
    assert it1[0] > 0 and it1[2] <= it1[1] and it0[0] > it1[0]          # the first call also evaluated the initial forces
    h.close()
