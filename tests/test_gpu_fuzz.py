"""-m gpu: seeded random configurations through the whole parity check (tree arrays bit for bit, list lengths bit
for bit, accelerations in tolerance; fused walk and hard-only walk, hard-step tree too).  Sizes, clustering, leaf and
group sizes, radii, opening criterion, grouping, changeover function and both readings of the hard list are drawn at
random, so the combinations no hand-written case names get exercised as well."""
import numpy as np
import pytest

from oracle import oracle as O
from workloads import CONFIGS

pytestmark = pytest.mark.gpu

from gpu_util import MAX_TOL, RMS_TOL, acc_errors, check_forces, compare_lists, compare_tree, make_hyb  # noqa: E402


def _random_case(seed):
    rng = np.random.default_rng(1000 + seed)
    n = int(rng.choice([1, 2, 3, 17, 64, 65, 333, 1000, 2049, 4097, 7001]))
    pos = np.zeros((n, 4), np.float32)
    nclump = int(rng.integers(1, 5))
    centres = rng.normal(size=(nclump, 3)) * rng.choice([0.1, 1.0, 30.0])
    scale = rng.choice([1e-3, 0.05, 1.0], size=nclump)
    which = rng.integers(0, nclump, size=n)
    pos[:, :3] = centres[which] + rng.normal(size=(n, 3)) * scale[which, None]
    if rng.random() < 0.3 and n > 40:                      # some coincident points (depth limit, chunked groups)
        k = int(rng.integers(2, 40)); i0 = int(rng.integers(0, n - k))
        pos[i0:i0 + k, :3] = pos[i0, :3]
    pos[:, 3] = rng.uniform(0.0 if rng.random() < 0.3 else 0.5, 2.0, n) / n
    vel = (rng.normal(size=(n, 4)) * 0.1).astype(np.float32); vel[:, 3] = 0
    leaf = int(rng.choice([1, 2, 4, 8, 16, 24]))
    group = int(rng.choice([g for g in (1, 4, 8, 16, 32, 48, 64) if g >= leaf]))
    r_out = float(rng.choice([0.003, 0.03, 0.3, 3.0]))
    over = dict(n=n, leaf_max=leaf, group_max=group, r_out=r_out, r_in=float(r_out * rng.choice([0.0, 0.1, 0.5])),
                theta=float(rng.choice([0.0, 0.3, 0.5, 0.8, 1.2])), eps=float(rng.choice([1e-3, 0.02])),
                mac=int(rng.integers(0, 2)), a_err=float(rng.choice([2.0 ** -8, 2.0 ** -4, 1e-6])),
                grouping=int(rng.integers(0, 3)), kfunc=int(rng.integers(0, 2)), hard_cut=int(rng.integers(0, 2)),
                hard_tree=int(rng.random() < 0.25), split=int(rng.random() < 0.85))
    return pos, vel, over


@pytest.mark.parametrize("seed", range(40))
def test_random_configuration(seed):
    pos, vel, over = _random_case(seed)
    cfg = CONFIGS[0].with_(**over)
    h = make_hyb(cfg, pos, vel)
    h.build_tree(); h.sync()
    t = O.Tree(pos, O.params_from(cfg))
    compare_tree(h, t, abs_mode=cfg.mac == 1)
    check_forces(h, t, split=cfg.split == 1)
    if cfg.split and not cfg.hard_tree:                    # the hard-step tree of hyb_step on the same store
        store = h.pos_m.cpu().numpy()
        h.build_tree_hard(); h.sync()
        gm = max(cfg.group_max // 2, cfg.leaf_max) if cfg.grouping == 2 else cfg.group_max
        th = O.Tree(store, O.params_from(cfg, group_max=gm))
        compare_tree(h, th, boxes_only=True)
        h.hard_force(); h.sync()
        compare_lists(h, th, O.MODE_HARD)
        a_s, a_h, _ = th.forces(O.MODE_HYBRID)
        rms, mx = acc_errors(h.a_hard.cpu().numpy()[:, :3], a_h, a_s + a_h)
        assert rms < RMS_TOL and mx < MAX_TOL, (rms, mx)
    store = h.pos_m.cpu().numpy()                          # once more on the same store: this fused walk follows the work
    h.build_tree(); h.sync()                               # order prepared from the first one's list lengths
    h.export("interactions")                               # (the counters run since the last read)
    check_forces(h, O.Tree(store, O.params_from(cfg)), split=cfg.split == 1)
    h.step(1); h.sync()
    assert np.all(np.isfinite(h.pos_m.cpu().numpy()))
    h.close()


@pytest.mark.parametrize("seed", range(4))
def test_random_configuration_medium(seed):
    """the same on both sides of the size where the walks change their work order and the hard walk its instantiation
    (3.8e5 particles on a B200), accelerations and list lengths on sampled groups"""
    from workloads import make_ic
    rng = np.random.default_rng(5000 + seed)
    n = int(rng.choice([378879, 378881, 400003, 524288]))
    kind = str(rng.choice(["plummer", "hernquist", "cold_sphere", "two_plummer"]))
    leaf = int(rng.choice([4, 8, 16, 24])); group = int(rng.choice([g for g in (16, 32, 48, 64) if g >= leaf]))
    r_out = float(rng.choice([0.01, 0.03, 0.08]))
    cfg = CONFIGS[2].with_(n=n, kind=kind, leaf_max=leaf, group_max=group, r_out=r_out, r_in=float(r_out * rng.choice([0.0, 0.1, 0.5])),
                           theta=float(rng.choice([0.4, 0.5, 0.8])), eps=float(rng.choice([1e-3, 0.01])), mac=int(rng.integers(0, 2)),
                           grouping=int(rng.integers(0, 3)), kfunc=int(rng.integers(0, 2)), hard_cut=int(rng.integers(0, 2)),
                           hard_tree=int(rng.random() < 0.3))
    pos, vel = make_ic(kind, n, 100 + seed)
    h = make_hyb(cfg, pos, vel)
    h.build_tree(); h.sync()
    t = O.Tree(pos, O.params_from(cfg))
    compare_tree(h, t, abs_mode=cfg.mac == 1)
    sample = lambda ng, k, s: np.sort(np.random.default_rng(s).choice(ng, size=min(k, ng), replace=False)).astype(np.int64)
    check_forces(h, t, gsel=sample(t.ng, 2048, seed))
    store = h.pos_m.cpu().numpy()                          # second walk on the same store: prepared work order
    h.build_tree(); h.sync(); h.export("interactions")
    t2 = O.Tree(store, O.params_from(cfg))
    check_forces(h, t2, gsel=sample(t2.ng, 1024, seed + 1))
    if not cfg.hard_tree:
        store = h.pos_m.cpu().numpy()
        h.build_tree_hard(); h.sync()
        gm = max(cfg.group_max // 2, cfg.leaf_max) if cfg.grouping == 2 else cfg.group_max
        th = O.Tree(store, O.params_from(cfg, group_max=gm))
        compare_tree(h, th, boxes_only=True)
        h.hard_force(); h.sync()
        compare_lists(h, th, O.MODE_HARD)
    h.step(1); h.sync()
    assert np.all(np.isfinite(h.pos_m.cpu().numpy()))
    h.close()
