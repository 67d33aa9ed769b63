"""Helpers shared by the -m gpu parity tests: run the CUDA path through the C-ABI binding and the
oracle on the same seeded inputs and compare stage by stage."""
import numpy as np

from oracle import oracle as O

TREE_INT = ("level", "first", "count", "child", "nchild", "parent", "level_offset")
RMS_TOL, MAX_TOL = 1e-5, 1e-4        # BASELINE.json north_star: relative to |a_total| per particle


def make_hyb(cfg, pos, vel, **over):
    import torch
    from paper_1406_6158_b200 import Hyb, HybParams
    P = HybParams.from_config(cfg, **over)
    dpos = torch.from_numpy(pos.copy()).cuda()
    dvel = torch.from_numpy(vel.copy()).cuda()
    return Hyb(P, dpos, dvel)


def compare_tree(h, t, abs_mode=False, boxes_only=False):
    """bit-exact comparison of every integer / fp32-decision output of a1-a7 (T2-T11).
    boxes_only: a hard-step tree (hyb_build_tree_hard) carries no moments and no opening radius."""
    c = h.export("counts")
    assert c[4] == 0, f"device status {c[4]}"
    assert (c[1], c[2]) == (t.nn, t.ng), (c, t.nn, t.ng)
    assert np.array_equal(h.export("bbox"), t.get("bbox"))
    assert np.array_equal(h.export("keys"), t.get("keys"))
    assert np.array_equal(h.export("perm"), t.get("perm"))
    assert np.array_equal(h.export("keys_sorted"), t.get("keys_sorted"))
    assert np.array_equal(h.pos_m.cpu().numpy(), t.get("pos_sorted"))
    for name in TREE_INT:
        assert np.array_equal(h.export(name), t.get(name)), name
    if not boxes_only:
        assert np.array_equal(h.export("com_m"), t.get("com_m"))
        assert np.array_equal(h.export("M64"), t.get("M64"))
        assert np.array_equal(h.export("C64"), t.get("C64"))
    assert np.array_equal(h.export("nlo")[:, :3], t.get("nlo"))
    assert np.array_equal(h.export("nhi")[:, :3], t.get("nhi"))
    if abs_mode:
        assert np.array_equal(h.export("B2"), t.get("B2"))
        assert np.array_equal(h.export("bmax"), t.get("bmax"))
    if not boxes_only:
        assert np.array_equal(h.export("ropen2"), t.get("ropen2"))
    assert np.array_equal(h.export("gfirst"), t.get("gfirst"))
    assert np.array_equal(h.export("gcount"), t.get("gcount"))
    assert np.array_equal(h.export("glo")[:, :3], t.get("glo"))
    assert np.array_equal(h.export("ghi")[:, :3], t.get("ghi"))


def compare_lists(h, t, mode, gsel=None):
    """list lengths per group (T13), bit-exact; gsel: only those groups (sampled check)."""
    nc, npart, nh = t.walk_counts(mode, gsel)
    sel = slice(None) if gsel is None else np.asarray(gsel)
    assert np.array_equal(h.export("ncell")[sel], nc)
    assert np.array_equal(h.export("npart")[sel], npart)
    assert np.array_equal(h.export("nhard")[sel], nh)


def acc_errors(a_gpu, a_ref, a_tot_ref):
    """rms and max of |a_gpu - a_ref| / |a_total_ref| over particles."""
    scale = np.linalg.norm(a_tot_ref, axis=1)
    diff = np.linalg.norm(a_gpu.astype(np.float64) - a_ref, axis=1)
    assert np.all(diff[scale == 0] == 0)             # an isolated particle feels exactly zero force
    err = np.where(scale > 0, diff / np.where(scale > 0, scale, 1.0), 0.0)
    return float(np.sqrt(np.mean(err ** 2))), float(err.max())


def check_forces(h, t, split=True, gsel=None, lists_full=True):
    """runs soft (and hard) force on the GPU and compares with the oracle (T14).
    gsel: accelerations only on those groups; lists_full=False: list lengths on gsel only."""
    mode = O.MODE_HYBRID if split else O.MODE_NORMAL
    h.soft_force()
    h.sync()
    lsel = None if lists_full else gsel
    compare_lists(h, t, mode, lsel)
    a_s, a_h, inter = t.forces(mode, gsel)
    gs = h.a_soft.cpu().numpy()[:, :3]; gh = h.a_hard.cpu().numpy()[:, :3]
    if gsel is not None:
        gf, gc = t.get("gfirst"), t.get("gcount")
        idx = np.concatenate([np.arange(gf[g], gf[g] + gc[g]) for g in gsel])
    else:
        idx = np.arange(t.n)
        got = h.export("interactions")
        assert (int(got[0]), int(got[1])) == (int(inter[0]), int(inter[1]))
    tot = a_s[idx] + a_h[idx]
    res = {"soft": acc_errors(gs[idx], a_s[idx], tot), "hard": acc_errors(gh[idx], a_h[idx], tot),
           "total": acc_errors(gs[idx] + gh[idx], tot, tot)}
    for k, (rms, mx) in res.items():
        assert rms < RMS_TOL and mx < MAX_TOL, (k, rms, mx)
    if split:
        h.a_hard.zero_()
        h.hard_force()
        h.sync()
        compare_lists(h, t, O.MODE_HARD, lsel)
        gh2 = h.a_hard.cpu().numpy()[:, :3]
        rms, mx = acc_errors(gh2[idx], a_h[idx], tot)
        assert rms < RMS_TOL and mx < MAX_TOL, ("hard-only", rms, mx)
        res["hard_only"] = (rms, mx)
    return res
