"""Pins for the virtual-domain LET counts (Eq. 14-15)."""
import numpy as np

from oracle import oracle as O
from workloads import CONFIGS, make_ic
from workloads.domains import virtual_domains


def _setup(n=6000, a_err=2.0 ** -8, r_out=0.2):
    cfg = CONFIGS[0].with_(n=n, mac=1, a_err=a_err, r_out=r_out, r_in=0.1 * r_out)
    pos, _ = make_ic(cfg.kind, cfg.n, 41)
    return cfg, pos, O.Tree(pos, O.params_from(cfg))


def _dist_to_box(x, lo, hi):
    d = np.maximum(0.0, np.maximum(lo - x, x - hi))
    return np.sqrt((d * d).sum(axis=1))


def test_domains_tile_space_and_balance():
    _, pos, _ = _setup()
    b = virtual_domains(pos, 2, 2, 2, seed=3)
    assert b.shape == (8, 6)
    inside = [(np.all(pos[:, :3] >= bb[:3], axis=1) & np.all(pos[:, :3] < bb[3:], axis=1)) for bb in b]
    assert np.array_equal(np.sum(inside, axis=0), np.ones(len(pos)))          # every particle in exactly one domain
    counts = np.array([m.sum() for m in inside])
    assert counts.min() > 0.5 * counts.mean() and counts.max() < 1.6 * counts.mean()


def test_local_counts_and_single_domain():
    cfg, pos, t = _setup()
    b = virtual_domains(pos, 2, 2, 2, seed=3)
    c = t.let_count(b)
    inside = np.array([(np.all(pos[:, :3] >= bb[:3], axis=1) & np.all(pos[:, :3] < bb[3:], axis=1)).sum() for bb in b])
    assert np.array_equal(c[:, 0], inside) and c[:, 0].sum() == cfg.n
    assert np.all(c[:, 2] <= c[:, 1]) and np.all(c[:, 1] > 0)
    whole = np.array([[-np.inf] * 3 + [np.inf] * 3], np.float32)
    assert np.array_equal(t.let_count(whole), [[cfg.n, 0, 0]])                  # one process: nothing to exchange


def test_everything_opened_is_brute_force():
    """a_err -> 0 makes r_b huge: every cell is opened, so every outside particle is sent one by one
    (N_soft = N - N_local) and the hard LET holds exactly the outside particles within R_2 of the domain"""
    cfg, pos, t = _setup(n=3000, a_err=1e-30, r_out=0.15)
    b = virtual_domains(pos, 2, 1, 2, seed=5)
    c = t.let_count(b)
    x = pos[:, :3].astype(np.float64)
    for j, bb in enumerate(b):
        lo, hi = bb[:3].astype(np.float64), bb[3:].astype(np.float64)
        ins = np.all(x >= lo, axis=1) & np.all(x < hi, axis=1)
        d = _dist_to_box(x[~ins], lo, hi)
        near = int((d < cfg.r_out * (1 - 1e-6)).sum()), int((d < cfg.r_out * (1 + 1e-6)).sum())
        assert c[j, 0] == ins.sum() and c[j, 1] == cfg.n - ins.sum()
        assert near[0] <= c[j, 2] <= near[1]


def test_cells_reduce_the_soft_let_and_cutoff_reduces_the_hard_let():
    cfg, pos, t = _setup(n=20000)
    b = virtual_domains(pos, 2, 2, 2, seed=7)
    c = t.let_count(b).astype(np.float64)
    assert np.all(c[:, 1] < 0.5 * (cfg.n - c[:, 0]))          # cells stand for many particles
    assert np.all(c[:, 2] < c[:, 1])                          # Eq. 15 only removes entries
    # a larger R_2 can only enlarge the hard LET
    t2 = O.Tree(pos, O.params_from(cfg.with_(r_out=2 * cfg.r_out)))
    assert np.all(t2.let_count(b)[:, 2] >= c[:, 2])
