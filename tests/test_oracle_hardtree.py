"""Pins for the paper-literal hard force (hard_tree = 1; the hard force is
computed by the tree algorithm too, with the traversal cut off for distant cells)."""
import numpy as np
import pytest

from oracle import oracle as O
from workloads import CONFIGS, make_ic


@pytest.fixture(scope="module")
def setup():
    cfg = CONFIGS[0].with_(n=3000, r_in=0.02, r_out=0.25, theta=0.6, hard_tree=1)
    pos, _ = make_ic(cfg.kind, cfg.n, 21)
    return cfg, pos, O.Tree(pos, O.params_from(cfg))


def test_split_is_exact_on_every_list_entry(setup):
    """K F + (1 - K) F = F for cells as for particles: the fused walk's soft + hard equals the plain
    normal-tree force on the same tree, and its lists are the normal tree's lists (no rule (b))."""
    cfg, pos, t = setup
    a_s, a_h, inter = t.forces(O.MODE_HYBRID)
    tn = O.Tree(pos, O.params_from(cfg, split=0))
    a_n, _, inter_n = tn.forces(O.MODE_NORMAL)
    scale = np.linalg.norm(a_n, axis=1)
    assert np.max(np.linalg.norm(a_s + a_h - a_n, axis=1) / scale) < 1e-12
    nc, npart, nh = t.walk_counts(O.MODE_HYBRID)
    ncn, npn, _ = tn.walk_counts(O.MODE_NORMAL)
    assert np.array_equal(nc, ncn) and np.array_equal(npart, npn)
    assert inter[0] == inter_n[0] and 0 < inter[1] < inter[0]
    assert np.linalg.norm(a_h, axis=1).max() > 0


def test_hard_only_walk_gives_the_hard_part_of_the_fused_walk(setup):
    """everything the cut-off drops is farther than r_out from every sink of the group, where K = 0"""
    cfg, pos, t = setup
    _, a_h, _ = t.forces(O.MODE_HYBRID)
    _, a_h2, _ = t.forces(O.MODE_HARD)
    assert np.max(np.abs(a_h2 - a_h)) <= 1e-13 * np.max(np.abs(a_h))
    assert np.array_equal(t.walk_counts(O.MODE_HARD)[2], t.walk_counts(O.MODE_HYBRID)[2])
    # the hard walk is much shorter than the soft walk: that is the point of the method
    nc_h, np_h, _ = t.walk_counts(O.MODE_HARD)
    nc_s, np_s, _ = t.walk_counts(O.MODE_HYBRID)
    assert (nc_h + np_h).sum() < 0.6 * (nc_s + np_s).sum()


def test_theta_zero_is_the_direct_hard_sum():
    cfg = CONFIGS[0].with_(n=700, theta=0.0, hard_tree=1, r_in=0.02, r_out=0.3)
    pos, _ = make_ic(cfg.kind, cfg.n, 22)
    t = O.Tree(pos, O.params_from(cfg))
    _, a_h, _ = t.forces(O.MODE_HARD)
    _, ah_direct, _ = O.direct(pos, cfg.G, cfg.eps, cfg.r_in, cfg.r_out)
    perm = t.get("perm")
    assert np.max(np.abs(a_h - ah_direct[perm])) < 1e-12 * np.max(np.abs(ah_direct))
    assert np.all(t.walk_counts(O.MODE_HARD)[0] == 0)


def test_tree_hard_force_approximates_the_direct_hard_sum(setup):
    """lower accuracy than the direct sum, but a tree-code error, not a different force"""
    cfg, pos, t = setup
    _, a_h, _ = t.forces(O.MODE_HARD)
    at, ah_direct, _ = O.direct(pos, cfg.G, cfg.eps, cfg.r_in, cfg.r_out)
    perm = t.get("perm")
    err = np.linalg.norm(a_h - ah_direct[perm], axis=1) / np.linalg.norm(at[perm], axis=1)
    assert 0 < err.max() < 3e-2 and np.sqrt(np.mean(err ** 2)) < 5e-3
    # and the direct-sum reading (hard_tree = 0) on the same particles is exact
    t0 = O.Tree(pos, O.params_from(cfg, hard_tree=0))
    _, a_h0, _ = t0.forces(O.MODE_HARD)
    assert np.max(np.abs(a_h0 - ah_direct[perm])) < 1e-12 * np.max(np.abs(ah_direct))
