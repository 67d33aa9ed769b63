"""-m gpu: the CUDA path (through the C-ABI) against the oracle, stage by stage."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from workloads import CONFIGS, make_ic

pytestmark = pytest.mark.gpu

from gpu_util import check_forces, compare_tree, make_hyb  # noqa: E402


def _run_case(cfg, pos, vel, **over):
    h = make_hyb(cfg, pos, vel, **over)
    h.build_tree()
    h.sync()
    t = O.Tree(pos, O.params_from(cfg, **over))
    compare_tree(h, t, abs_mode=over.get("mac", cfg.mac) == 1)
    res = check_forces(h, t, split=over.get("split", cfg.split) == 1)
    h.close()
    return res


@pytest.mark.parametrize("hard_cut", [1, 0])
@pytest.mark.parametrize("grouping", [1, 0])
@pytest.mark.parametrize("mac", [0, 1])
def test_cfg0_all_stages(mac, grouping, hard_cut):
    cfg = CONFIGS[0]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    print(_run_case(cfg, pos, vel, mac=mac, grouping=grouping, hard_cut=hard_cut))


def test_cfg0_normal_tree():
    cfg = CONFIGS[0]
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    print(_run_case(cfg, pos, vel, split=0))


@pytest.mark.parametrize("n,kind,leaf,group", [(20011, "plummer", 16, 64), (9973, "hernquist", 8, 32),
                                               (33333, "cold_sphere", 16, 64), (5000, "two_plummer", 1, 1),
                                               (1, "cold_sphere", 8, 32), (2, "cold_sphere", 8, 32),
                                               (37, "plummer", 8, 32)])
def test_ragged_sizes(n, kind, leaf, group):
    for grouping, hard_cut in ((1, 1), (0, 1), (1, 0)):
        cfg = CONFIGS[1].with_(n=n, kind=kind, leaf_max=leaf, group_max=group, grouping=grouping, hard_cut=hard_cut)
        pos, vel = make_ic(kind, n, 17)
        print(_run_case(cfg, pos, vel))


def test_coincident_points_and_depth_limit():
    cfg = CONFIGS[0].with_(leaf_max=4, group_max=8)
    rng = np.random.default_rng(2)
    pos = np.zeros((3000, 4), np.float32)
    pos[:, :3] = rng.normal(size=(3000, 3))
    pos[100:400, :3] = pos[100, :3]                # 300 coincident points -> level-21 leaf, chunked groups
    pos[500:520, :3] = pos[500, :3]
    pos[:, 3] = 1.0 / 3000
    vel = np.zeros_like(pos)
    print(_run_case(cfg, pos, vel))
    print(_run_case(cfg, pos, vel, grouping=0))
    print(_run_case(cfg, pos, vel, hard_cut=0))


def test_theta_zero_opens_everything():
    cfg = CONFIGS[0].with_(n=1500, theta=0.0)
    pos, vel = make_ic("plummer", 1500, 3)
    h = make_hyb(cfg, pos, vel)
    h.build_tree(); h.soft_force(); h.sync()
    assert np.all(h.export("ncell") == 0) and np.all(h.export("npart") == 1500)
    at, ah, as_ = O.direct(pos, cfg.G, cfg.eps, cfg.r_in, cfg.r_out)
    perm = h.export("perm")
    tot = (h.a_soft + h.a_hard).cpu().numpy()[:, :3]
    err = np.linalg.norm(tot - at[perm], axis=1) / np.linalg.norm(at[perm], axis=1)
    assert err.max() < 1e-4 and np.sqrt(np.mean(err ** 2)) < 1e-5
    h.close()


def test_poly7_changeover_function():
    """north_star's alternative K (HYB_K_POLY7, R6): same lists, different split of the pair force."""
    for cfg, seed in ((CONFIGS[0], 0), (CONFIGS[1].with_(n=30011), 9)):
        pos, vel = make_ic(cfg.kind, cfg.n, seed)
        res = _run_case(cfg, pos, vel, kfunc=1)
        res0 = _run_case(cfg, pos, vel, kfunc=0)
        print(res)
        assert res["hard"] != res0["hard"]                 # the two changeover functions really differ


def test_paper_parameter_recipe():
    """the paper's own parameter choice: eps = 0.1 N^-0.26, R1 = 1.03 N^-1/3, R2 = 2 R1,
    absolute MAC with a_err = 2^-8, n = 4."""
    from workloads import paper_params
    cfg = paper_params(1 << 16, seed=12)
    pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
    print(_run_case(cfg, pos, vel))
    h = make_hyb(cfg, pos, vel)
    h.step(1); h.sync()
    assert np.all(np.isfinite(h.pos_m.cpu().numpy()))
    h.close()


def test_error_paths_on_device():
    """every failure is reported as an error code, never silently (include/hyb.h)"""
    import torch
    from paper_1406_6158_b200 import Hyb, HybError, HybParams
    cfg = CONFIGS[0].with_(n=1000)
    pos, vel = make_ic(cfg.kind, cfg.n, 4)
    # force call without a tree
    h = make_hyb(cfg, pos, vel)
    with pytest.raises(HybError) as ei:
        h.hard_force()
    assert ei.value.code == -5
    with pytest.raises(HybError) as ei:
        h.soft_force()
    assert ei.value.code == -5
    h.build_tree(); h.soft_force(); h.sync()
    # parameters that cannot change after init
    with pytest.raises(HybError) as ei:
        h.set_params(HybParams.from_config(cfg, leaf_max=4))
    assert ei.value.code == -1
    # changing theta invalidates the tree
    h.set_params(HybParams.from_config(cfg, theta=0.7))
    with pytest.raises(HybError) as ei:
        h.soft_force()
    assert ei.value.code == -5
    h.close()
    # non-finite position, negative mass
    for bad in ("nan", "neg"):
        p2 = pos.copy()
        if bad == "nan":
            p2[17, 1] = np.nan
        else:
            p2[5, 3] = -1.0
        h = make_hyb(cfg, p2, vel)
        h.build_tree()
        with pytest.raises(HybError) as ei:
            h.sync()
        assert ei.value.code == -3
        h.close()
    # misaligned / missing pointers and a workspace that is too small are refused by hyb_init
    from paper_1406_6158_b200.binding import hyb_workspace_bytes, lib
    import ctypes as C
    P = HybParams.from_config(cfg)
    need = hyb_workspace_bytes(cfg.n, P)
    dpos = torch.from_numpy(pos).cuda(); dvel = torch.from_numpy(vel).cuda()
    acc = torch.zeros_like(dpos); ids = torch.arange(cfg.n, dtype=torch.int32, device="cuda")
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    hnd = C.c_void_p()
    rc = lib().hyb_init(C.byref(hnd), C.byref(P), cfg.n, dpos.data_ptr(), dvel.data_ptr(), acc.data_ptr(), acc.data_ptr(),
                        ids.data_ptr(), ws.data_ptr(), need - 1, 0, None)
    assert rc == -2 and not hnd.value
    rc = lib().hyb_init(C.byref(hnd), C.byref(P), cfg.n, dpos.data_ptr() + 4, dvel.data_ptr(), acc.data_ptr(), acc.data_ptr(),
                        ids.data_ptr(), ws.data_ptr(), need, 0, None)
    assert rc == -1 and not hnd.value


@pytest.mark.parametrize("hard_cut", [1, 0])
@pytest.mark.parametrize("kfunc", [0, 1])
def test_paper_literal_hard_walk(kfunc, hard_cut):
    """hard_tree = 1: MAC-approximated hard force, K-weighted cells"""
    for cfg, seed in ((CONFIGS[0].with_(r_out=0.25, r_in=0.02, theta=0.6), 0), (CONFIGS[1].with_(n=40013, r_out=0.15), 9),
                      (CONFIGS[0].with_(n=777, theta=0.0), 3)):
        pos, vel = make_ic(cfg.kind, cfg.n, seed)
        print(_run_case(cfg, pos, vel, hard_tree=1, kfunc=kfunc, hard_cut=hard_cut))
    cfg = CONFIGS[0].with_(hard_tree=1, r_out=0.2)
    pos, vel = make_ic(cfg.kind, cfg.n, 5)
    h = make_hyb(cfg, pos, vel)
    h.step(2); h.sync()
    assert np.all(np.isfinite(h.pos_m.cpu().numpy()))
    h.close()


@pytest.mark.parametrize("case", ["one_point", "zero_masses", "collinear", "far_offset", "two_clumps"])
def test_degenerate_inputs(case):
    """the degenerate inputs the method has: a zero-size root cube, massless particles and cells, a tree that
    is a chain, coordinates with few significant bits left for the separations, an almost empty root cube"""
    rng = np.random.default_rng(7)
    n = 700
    pos = np.zeros((n, 4), np.float32)
    pos[:, 3] = 1.0 / n
    if case == "one_point":
        pos[:, :3] = np.float32(0.25)
    elif case == "zero_masses":
        pos[:, :3] = rng.normal(size=(n, 3))
        pos[::3, 3] = 0.0
        pos[300:340, 3] = 0.0                      # whole leaves without mass: COM falls back to the box corner (T9)
    elif case == "collinear":
        pos[:, 0] = np.sort(rng.uniform(-1, 1, n)); pos[:, 1] = 0.5; pos[:, 2] = -0.25
    elif case == "far_offset":
        pos[:, :3] = 1000.0 + 0.05 * rng.normal(size=(n, 3))
    else:
        pos[: n // 2, :3] = 1e-3 * rng.normal(size=(n // 2, 3))
        pos[n // 2:, :3] = 50.0 + 1e-3 * rng.normal(size=(n - n // 2, 3))
    vel = np.zeros_like(pos)
    cfg = CONFIGS[0].with_(n=n, r_in=0.002, r_out=0.02) if case in ("far_offset", "two_clumps") else CONFIGS[0].with_(n=n)
    for mac in (0, 1):
        print(case, mac, _run_case(cfg, pos, vel, mac=mac))


def test_bitwise_reproducible():
    """work is handed out by atomic counters, but every sum has a fixed order: two runs agree bit for bit"""
    cfg = CONFIGS[1].with_(n=60013)
    pos, vel = make_ic(cfg.kind, cfg.n, 77)
    outs = []
    for _ in range(2):
        h = make_hyb(cfg, pos, vel)
        h.step(2); h.sync()
        outs.append([t.cpu().numpy().copy() for t in (h.pos_m, h.vel, h.a_soft, h.a_hard, h.ids)])
        h.close()
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


def test_hard_walk_work_order_paths_agree():
    """The work order of a hard walk (heavy groups cut into sink ranges, chosen from the list lengths of the
    previous walk) is prepared by the tree build for the first walk after it and by split_kernel for any
    further walk on the same tree; the two counter slots alternate between launches.  The lists never
    change; the sums are bit-identical whenever the same groups are cut, and differ only in rounding
    when the cut set differs (a range of fewer sinks combines its partial sums in another order)."""
    cfg = CONFIGS[2].with_(n=150001)                        # Hernquist cusp: some groups are heavy enough to be cut
    pos, vel = make_ic(cfg.kind, cfg.n, 9)
    h = make_hyb(cfg, pos, vel)

    def close(a, b):
        return float((a - b).norm() / b.norm()) < 1e-6

    h.build_tree(); h.hard_force(); h.sync()                 # no previous walk: nothing is cut
    first = h.a_hard.clone()
    nh = h.export("nhard").copy()
    h.hard_force(); h.sync()                                 # split_kernel, estimates from the first walk
    second = h.a_hard.clone()
    assert np.array_equal(nh, h.export("nhard")) and close(second, first)
    for _ in range(3):                                       # same estimates, both counter slots
        h.hard_force(); h.sync()
        assert torch.equal(second, h.a_hard)
        assert np.array_equal(nh, h.export("nhard"))
    h.soft_force(); h.sync()                                 # fused walk: the same lists, another summation order
    assert close(h.a_hard, first)
    h.hard_force(); h.sync()
    assert torch.equal(second, h.a_hard)
    h.step(1); h.build_tree(); h.hard_force(); h.sync()      # after a step: the build prepares the order
    again = h.a_hard.clone()
    nh2 = h.export("nhard").copy()
    h.hard_force(); h.sync()
    assert np.array_equal(nh2, h.export("nhard")) and close(h.a_hard, again)
    h.close()
