"""-m gpu: the five BASELINE.json configurations at FULL size through the C-ABI against the oracle.

Tree, ordering, node and group arrays and list lengths are compared bit for bit over the whole
problem (cfg4: list lengths in full at the centre sweep point, on a seeded sample of groups at the
others); accelerations on all particles up to N = 2^20 and on a seeded sample of sink groups above
(an fp64 evaluation of every group at 2^24 for nine sweep points does not finish in
minutes on the host cores).  Multi-step parity is by snapshot: after hyb_step the oracle is fed the
GPU's current fp32 store, because fp32 and fp64 trajectories legitimately diverge."""
import numpy as np
import pytest

from oracle import oracle as O
from workloads import CONFIGS, make_ic
from workloads.configs import CFG4_ROUTS, CFG4_THETAS

pytestmark = pytest.mark.gpu

from gpu_util import acc_errors, check_forces, compare_lists, compare_tree, make_hyb, MAX_TOL, RMS_TOL  # noqa: E402


def _sample_groups(ng, k, seed):
    rng = np.random.default_rng(seed)
    return np.sort(rng.choice(ng, size=min(k, ng), replace=False)).astype(np.int64)


@pytest.mark.parametrize("mac", [0, 1])
def test_cfg1_full(mac):
    cfg = CONFIGS[1]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel, mac=mac)
    h.build_tree(); h.sync()
    t = O.Tree(pos, O.params_from(cfg, mac=mac))
    compare_tree(h, t, abs_mode=mac == 1)
    print(check_forces(h, t))
    h.close()


@pytest.mark.parametrize("mac,hard_cut", [(0, 1), (1, 1), (0, 0)])
def test_cfg2_full(mac, hard_cut):
    """the configuration bench.py times (N = 2^20 Hernquist), every particle; both readings of the hard list (R30)."""
    cfg = CONFIGS[2].with_(hard_cut=hard_cut)
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel, mac=mac)
    h.build_tree(); h.sync()
    t = O.Tree(pos, O.params_from(cfg, mac=mac))
    compare_tree(h, t, abs_mode=mac == 1)
    print(check_forces(h, t))
    h.close()


def test_cfg2_single_node_groups():
    """the other reading of R17 (one tree node per sink group) at the benchmark size"""
    cfg = CONFIGS[2]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel, grouping=0)
    h.build_tree(); h.sync()
    t = O.Tree(pos, O.params_from(cfg, grouping=0))
    compare_tree(h, t)
    print(check_forces(h, t, gsel=_sample_groups(t.ng, 8192, 8)))
    h.close()


def test_cfg2_paper_literal_hard_walk():
    """hard_tree = 1 at the benchmark size: lists in full, accelerations on a sample of groups"""
    cfg = CONFIGS[2]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel, hard_tree=1)
    h.build_tree(); h.sync()
    t = O.Tree(pos, O.params_from(cfg, hard_tree=1))
    compare_tree(h, t)
    print(check_forces(h, t, gsel=_sample_groups(t.ng, 4096, 9)))
    h.close()


def test_cfg2_normal_tree():
    cfg = CONFIGS[2]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel, split=0)
    h.build_tree(); h.sync()
    t = O.Tree(pos, O.params_from(cfg, split=0))
    compare_tree(h, t)
    print(check_forces(h, t, split=False, gsel=_sample_groups(t.ng, 8192, 5)))
    h.close()


@pytest.mark.parametrize("mac", [0, 1])
def test_cfg3_full_tree_sampled_forces(mac):
    cfg = CONFIGS[3]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel, mac=mac)
    h.build_tree(); h.sync()
    t = O.Tree(pos, O.params_from(cfg, mac=mac))
    compare_tree(h, t, abs_mode=mac == 1)
    print(check_forces(h, t, gsel=_sample_groups(t.ng, 8192, 6)))
    h.close()


def test_cfg4_sweep():
    """N = 2^24 two-Plummer merger, theta x r_out sweep (r_in = 0.1 r_out) on one context via
    hyb_set_params; the store stays in the order the first build left it, so every later build
    (and its oracle tree) starts from that order."""
    cfg = CONFIGS[4]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel)
    from paper_1406_6158_b200 import HybParams
    first = True
    for theta in CFG4_THETAS:
        for r_out in CFG4_ROUTS:
            over = dict(theta=theta, r_out=r_out, r_in=0.1 * r_out)
            centre = theta == 0.5 and r_out == 0.01
            h.set_params(HybParams.from_config(cfg, **over))
            store = h.pos_m.cpu().numpy()            # input order of this build
            h.build_tree(); h.sync()
            t = O.Tree(store, O.params_from(cfg, **over))
            if first or centre:
                compare_tree(h, t)
            else:                                     # same particles: the parts that depend on the point
                c = h.export("counts")
                assert (c[1], c[2], c[4]) == (t.nn, t.ng, 0)
                assert np.array_equal(h.export("perm"), t.get("perm"))
                assert np.array_equal(h.export("ropen2"), t.get("ropen2"))
                assert np.array_equal(h.export("com_m"), t.get("com_m"))
            gsel = _sample_groups(t.ng, 8192, 7)
            res = check_forces(h, t, gsel=gsel[::8], lists_full=False)
            compare_lists(h, t, O.MODE_HARD, None if centre else gsel)
            h.soft_force(); h.sync()
            compare_lists(h, t, O.MODE_HYBRID, None if centre else gsel)
            print(over, res)
            first = False
            del t
    h.close()


def test_cfg4_absolute_mac():
    """the paper's own opening criterion (Eq. 5-6, a_err = 2^-8) at N = 2^24, centre sweep point"""
    cfg = CONFIGS[4].with_(mac=1)
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel)
    h.build_tree(); h.sync()
    t = O.Tree(pos, O.params_from(cfg))
    compare_tree(h, t, abs_mode=True)
    gsel = _sample_groups(t.ng, 4096, 13)
    print(check_forces(h, t, gsel=gsel[::4], lists_full=False))
    h.close()


def _snapshot_parity(h, cfg, gsel_k=None):
    """forces the GPU left after hyb_step vs the oracle on the GPU's own current store."""
    h.sync()
    store = h.pos_m.cpu().numpy()
    t = O.Tree(store, O.params_from(cfg))
    # the store is already in Morton order: the oracle's permutation must be the identity
    assert np.array_equal(t.get("perm"), np.arange(cfg.n, dtype=np.uint32))
    assert np.array_equal(h.export("keys_sorted"), t.get("keys_sorted"))
    for name in ("level", "first", "count", "child", "nchild", "parent", "com_m", "ropen2", "gfirst", "gcount"):
        assert np.array_equal(h.export(name), t.get(name)), name
    gsel = None if gsel_k is None else _sample_groups(t.ng, gsel_k, 11)
    a_s, a_h, _ = t.forces(O.MODE_HYBRID, gsel)
    if gsel is None:
        idx = np.arange(cfg.n)
    else:
        gf, gc = t.get("gfirst"), t.get("gcount")
        idx = np.concatenate([np.arange(gf[g], gf[g] + gc[g]) for g in gsel])
    gs = h.a_soft.cpu().numpy()[idx, :3]; gh = h.a_hard.cpu().numpy()[idx, :3]
    tot = a_s[idx] + a_h[idx]
    res = {"soft": acc_errors(gs, a_s[idx], tot), "hard": acc_errors(gh, a_h[idx], tot)}
    for k, (rms, mx) in res.items():
        assert rms < RMS_TOL and mx < MAX_TOL, (k, rms, mx)
    return res


def test_cfg0_steps_energy_and_snapshot():
    """config 0 as written: 64 soft steps of 4 hard subcycles; energy drift bound is ours (R23)."""
    cfg = CONFIGS[0]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    m = pos[:, 3].copy()
    k0, w0 = O.energy(pos[:, :3], vel[:, :3], m, cfg.G, cfg.eps)
    h = make_hyb(cfg, pos, vel)
    h.step(cfg.n_soft_steps)
    print(_snapshot_parity(h, cfg))
    x = h.pos_m.cpu().numpy(); v = h.vel.cpu().numpy()
    ids = h.ids.cpu().numpy()
    assert np.array_equal(np.sort(ids), np.arange(cfg.n))           # id tracks the permutation
    assert np.array_equal(x[:, 3], m[ids])
    k1, w1 = O.energy(x[:, :3], v[:, :3], x[:, 3].copy(), cfg.G, cfg.eps)
    drift = abs((k1 + w1) - (k0 + w0)) / abs(k0 + w0)
    print("energy drift", drift)
    assert drift < 1e-3
    # momentum: the hard part is pairwise antisymmetric, the tree part is not exactly
    p = (x[:, 3:4].astype(np.float64) * v[:, :3]).sum(0)
    assert np.abs(p).max() < 1e-4
    h.close()


@pytest.mark.parametrize("ci,gsel_k", [(1, None), (2, 4096)])
def test_steps_snapshot(ci, gsel_k):
    cfg = CONFIGS[ci]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel)
    h.step(2)
    print(_snapshot_parity(h, cfg, gsel_k))
    h.close()


def test_step_matches_oracle_step_short():
    """one soft cycle from the same state: fp32 GPU vs fp64 oracle trajectories agree to fp32 accuracy."""
    cfg = CONFIGS[0]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    h = make_hyb(cfg, pos, vel)
    h.step(1); h.sync()
    ids = h.ids.cpu().numpy().astype(np.int64)
    xg = np.empty((cfg.n, 3)); vg = np.empty((cfg.n, 3))
    xg[ids] = h.pos_m.cpu().numpy()[:, :3]; vg[ids] = h.vel.cpu().numpy()[:, :3]
    x = pos[:, :3].astype(np.float64).copy(); v = vel[:, :3].astype(np.float64).copy()
    O.step(x, v, pos[:, 3], O.params_from(cfg), 1)
    assert np.abs(xg - x).max() < 2e-6 and np.abs(vg - v).max() < 2e-5
    h.close()
