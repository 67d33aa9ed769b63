"""Pins for the particle-level cut of the hard list (hard_cut = 1, R30).

PAPER.md:76, 82-85: F_hard = K(r) F and K(r) = 0 for r >= R_2; the hard force is cut
off beyond R_2.  With hard_cut = 1 the hard list of a sink group holds exactly the particles that are
within r_out of the group's box.  That set has a plain definition that needs no tree at all, so the pin is
brute force over ALL particles; and because only particles with K = 0 for every sink are dropped, the
hard force must not change."""
import numpy as np
import pytest

from oracle import oracle as O
from workloads import CONFIGS, make_ic

F = np.float32


def _brute_force_list(ps, glo, ghi, r_out):
    """{ j : fp32 distance^2 from x_j to the box [glo, ghi] < r_out^2 }, over every particle"""
    x = ps[:, :3].astype(F)
    e = np.maximum(F(0), np.maximum(glo[None, :].astype(F) - x, x - ghi[None, :].astype(F))).astype(F)
    d2 = (e[:, 0] * e[:, 0] + e[:, 1] * e[:, 1]) + e[:, 2] * e[:, 2]
    return set(np.nonzero(d2 < F(r_out) * F(r_out))[0].tolist())


@pytest.mark.parametrize("grouping,mac", [(1, 0), (0, 0), (1, 1)])
def test_hard_list_is_the_brute_force_set(grouping, mac):
    cfg = CONFIGS[0].with_(hard_cut=1, grouping=grouping, mac=mac)
    pos, _ = make_ic(cfg.kind, cfg.n, cfg.seed)
    t = O.Tree(pos, O.params_from(cfg))
    t0 = O.Tree(pos, O.params_from(cfg, hard_cut=0))
    ps, glo, ghi = t.get("pos_sorted"), t.get("glo"), t.get("ghi")
    gf, gc = t.get("gfirst"), t.get("gcount")
    nc, npart, nh = t.walk_counts(O.MODE_HYBRID)
    nc_h, np_h, nh_h = t.walk_counts(O.MODE_HARD)
    nc0, np0, nh0 = t0.walk_counts(O.MODE_HYBRID)
    # the cut changes nothing but the hard list: same cells, same particle list, hard walk == fused walk
    assert np.array_equal(nc, nc0) and np.array_equal(npart, np0) and np.array_equal(nh, nh_h)
    assert np.array_equal(np_h, nh0) and np.all(nc_h == 0)           # a hard walk opens the leaves within r_out, nothing else
    assert np.all(nh <= nh0) and nh.sum() < 0.8 * nh0.sum() and np.all(nh >= gc)
    x64 = ps[:, :3].astype(np.float64)
    for g in range(0, t.ng, 3):
        want = _brute_force_list(ps, glo[g], ghi[g], cfg.r_out)
        for mode in (O.MODE_HYBRID, O.MODE_HARD):
            _, parts, hard = t.walk_lists(mode, g)
            assert set(parts[hard].tolist()) == want
        assert nh[g] == len(want)
        _, parts0, hard0 = t0.walk_lists(O.MODE_HARD, g)
        assert want <= set(parts0[hard0].tolist())                        # a subset of the leaf-level list
        # and a superset of the true neighbours of the group's sinks (exact distances)
        mem = x64[gf[g]:gf[g] + gc[g]]
        d = np.sqrt(((x64[None, :, :] - mem[:, None, :]) ** 2).sum(axis=2)).min(axis=0)
        assert set(np.nonzero(d < cfg.r_out * (1 - 1e-6))[0].tolist()) <= want


def test_hard_force_does_not_change():
    """what the cut drops carries K = 0 for every sink of the group (Eq. 10: Y <= 0)"""
    cfg = CONFIGS[0]
    pos, _ = make_ic(cfg.kind, cfg.n, cfg.seed)
    t1 = O.Tree(pos, O.params_from(cfg, hard_cut=1))
    t0 = O.Tree(pos, O.params_from(cfg, hard_cut=0))
    for mode in (O.MODE_HYBRID, O.MODE_HARD):
        s1, h1, i1 = t1.forces(mode)
        s0, h0, i0 = t0.forces(mode)
        scale = np.abs(h0).max()
        assert np.abs(h1 - h0).max() <= 1e-15 * scale and np.array_equal(s1, s0)
        assert i1[0] == i0[0] and i1[1] < 0.8 * i0[1]
    perm = t1.get("perm")
    _, ah, _ = O.direct(pos, cfg.G, cfg.eps, cfg.r_in, cfg.r_out)
    assert np.abs(h1 - ah[perm]).max() < 1e-13                               # still the exact direct hard sum (R20)
    nh = t1.walk_counts(O.MODE_HARD)[2].astype(np.int64)
    assert i1[1] == float(nh @ t1.get("gcount").astype(np.int64))


def test_cut_with_the_paper_literal_hard_walk():
    """hard_tree = 1: near cells are kept whole, particles of opened near leaves are cut"""
    cfg = CONFIGS[0].with_(n=3000, r_in=0.02, r_out=0.25, theta=0.6, hard_tree=1)
    pos, _ = make_ic(cfg.kind, cfg.n, 21)
    t1 = O.Tree(pos, O.params_from(cfg, hard_cut=1))
    t0 = O.Tree(pos, O.params_from(cfg, hard_cut=0))
    s1, h1, _ = t1.forces(O.MODE_HYBRID)
    s0, h0, _ = t0.forces(O.MODE_HYBRID)
    assert np.abs(h1 - h0).max() <= 1e-15 * np.abs(h0).max() and np.array_equal(s1, s0)
    c1, c0 = t1.walk_counts(O.MODE_HYBRID), t0.walk_counts(O.MODE_HYBRID)
    assert np.array_equal(c1[0], c0[0]) and np.array_equal(c1[1], c0[1]) and np.all(c1[2] <= c0[2])
    assert np.array_equal(t1.walk_counts(O.MODE_HARD)[2], c1[2])
