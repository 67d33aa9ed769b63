"""Pins for the oracle's forces (T14) -- closed forms, brute force, conservation, analytic profiles."""
import numpy as np
import pytest

from oracle import oracle as O
from workloads import make_ic
from test_oracle_formulas import _params


def test_two_body_closed_form():
    # PAPER.md:35 Eq. 2 and Eq. 7-9: a_1 = G m_2 d / (d^2 + eps^2)^{3/2}, hard = K(d) a_1, soft = (1-K(d)) a_1
    G, eps, r_in, r_out = 2.5, 0.05, 0.1, 0.4
    for d in (0.05, 0.1, 0.17, 0.25, 0.33, 0.4, 0.9):
        p = np.array([[0.1, 0.2, 0.3, 3.0], [0.1 + d, 0.2, 0.3, 5.0]], np.float32)
        dd = float(p[1, 0]) - float(p[0, 0])
        t = O.Tree(p, _params(G=G, eps=eps, r_in=r_in, r_out=r_out))
        a_s, a_h, inter = t.forces(O.MODE_HYBRID)
        perm = t.get("perm")
        a_s, a_h = a_s[np.argsort(perm)], a_h[np.argsort(perm)]
        Y = (float(np.float32(r_out)) - dd) / (float(np.float32(r_out)) - float(np.float32(r_in)))
        Kd = 1.0 if Y >= 1 else 0.0 if Y <= 0 else 10 * Y ** 6 - 15 * Y ** 8 + 6 * Y ** 10
        s = float(np.float32(G)) / (dd * dd + float(np.float32(eps)) ** 2) ** 1.5
        a1, a2 = 5.0 * s * dd, -3.0 * s * dd
        assert a_h[0, 0] == pytest.approx(Kd * a1, rel=1e-12, abs=1e-14)
        assert a_s[0, 0] == pytest.approx((1 - Kd) * a1, rel=1e-12, abs=1e-14)
        assert a_h[1, 0] == pytest.approx(Kd * a2, rel=1e-12, abs=1e-14)
        assert a_s[1, 0] == pytest.approx((1 - Kd) * a2, rel=1e-12, abs=1e-14)
        assert np.all(a_s[:, 1:] == 0) and np.all(a_h[:, 1:] == 0)
        at, ah, as_ = O.direct(p, G, eps, r_in, r_out)
        assert at[0, 0] == pytest.approx(a1, rel=1e-13) and ah[0, 0] == pytest.approx(Kd * a1, rel=1e-12, abs=1e-14)


def _numpy_direct(p, G, eps):
    x = p[:, :3].astype(np.float64); m = p[:, 3].astype(np.float64)
    d = x[None, :, :] - x[:, None, :]
    r2 = (d ** 2).sum(axis=2) + float(np.float32(eps)) ** 2
    w = m[None, :] / r2 ** 1.5
    np.fill_diagonal(w, 0.0)
    return float(np.float32(G)) * (w[:, :, None] * d).sum(axis=1)


def test_direct_matches_numpy_definition():
    rng = np.random.default_rng(0)
    p = rng.normal(size=(300, 4)).astype(np.float32); p[:, 3] = rng.uniform(0.5, 2, 300)
    at, ah, as_ = O.direct(p, 1.3, 0.07, 0.1, 0.5)
    assert np.allclose(at, _numpy_direct(p, 1.3, 0.07), rtol=1e-12, atol=1e-13)
    assert np.allclose(ah + as_, at, rtol=1e-13, atol=1e-12)                    # Eq. 7


def test_theta0_hard_plus_soft_is_direct(cfg0, ic0):
    t = O.Tree(ic0[0], O.params_from(cfg0, theta=0.0))
    a_s, a_h, inter = t.forces(O.MODE_HYBRID)
    perm = t.get("perm")
    at, ah, as_ = O.direct(ic0[0], cfg0.G, cfg0.eps, cfg0.r_in, cfg0.r_out)
    assert np.abs(a_s + a_h - at[perm]).max() < 1e-13 * np.abs(at).max() * 10
    assert np.abs(a_h - ah[perm]).max() < 1e-13 and np.abs(a_s - as_[perm]).max() < 1e-12
    assert inter == (float(cfg0.n) ** 2, pytest.approx(float(t.walk_counts(0)[2].astype(np.int64) @ t.get("gcount"))))


def test_hard_sum_is_exact_at_any_theta_and_conserves_momentum(tree0, cfg0, ic0):
    a_s, a_h, _ = tree0.forces(O.MODE_HYBRID)
    a_s2, a_h2, _ = tree0.forces(O.MODE_HARD)
    assert np.array_equal(a_h, a_h2) and np.all(a_s2 == 0)
    perm = tree0.get("perm")
    at, ah, as_ = O.direct(ic0[0], cfg0.G, cfg0.eps, cfg0.r_in, cfg0.r_out)
    assert np.abs(a_h - ah[perm]).max() < 1e-13                               # R20: exact K-weighted direct sum
    m = tree0.get("pos_sorted")[:, 3].astype(np.float64)
    mom = (m[:, None] * a_h).sum(axis=0)                                      # Newton's third law, K symmetric
    assert np.abs(mom).max() < 1e-15 * np.abs(m[:, None] * a_h).sum()
    # tree error of the total at theta = 0.5: sanity, ~1e-3
    err = np.linalg.norm(a_s + a_h - at[perm], axis=1) / np.linalg.norm(at[perm], axis=1)
    assert 1e-5 < err.mean() < 5e-3
    a_n, _, _ = tree0.forces(O.MODE_NORMAL)
    errn = np.linalg.norm(a_n - at[perm], axis=1) / np.linalg.norm(at[perm], axis=1)
    assert 1e-5 < errn.mean() < 5e-3


def test_abs_mac_accuracy(cfg0, ic0):
    # a_err controls the monopole error of every accepted cell (absolute, in units of
    # acceleration / G); the summed error scales with it.  Sanity, not a pin of Eq. 5 (see test_rb_*).
    at, _, _ = O.direct(ic0[0], cfg0.G, cfg0.eps, cfg0.r_in, cfg0.r_out)
    errs = []
    for a_err in (2.0 ** -8, 2.0 ** -12):
        t = O.Tree(ic0[0], O.params_from(cfg0, mac=1, a_err=a_err))
        a_s, a_h, _ = t.forces(O.MODE_HYBRID)
        err = np.linalg.norm(a_s + a_h - at[t.get("perm")], axis=1)
        assert err.max() < 4 * a_err and err.mean() < a_err
        errs.append(err.mean())
    assert errs[1] < errs[0] / 4


def _radial_profile(kind, n, seed, edges, eps=0.002, theta=0.4):
    p, _ = make_ic(kind, n, seed)
    t = O.Tree(p, _params(eps=eps, theta=theta, leaf_max=16, group_max=64, r_in=0.003, r_out=0.03))
    a_s, a_h, _ = t.forces(O.MODE_HYBRID)
    x = t.get("pos_sorted")[:, :3].astype(np.float64)
    # the generators recentre on the sample COM (a large shift for Hernquist's heavy tail): measure
    # about the coordinate-wise median, a robust estimate of the density centre
    x = x - np.median(x, axis=0)
    r = np.linalg.norm(x, axis=1)
    ar = ((a_s + a_h) * x).sum(axis=1) / r
    out = []
    for lo, hi in zip(edges[:-1], edges[1:]):
        msk = (r >= lo) & (r < hi)
        out.append((np.mean(r[msk]), np.mean(ar[msk]), msk.sum(), r[msk], ar[msk]))
    return out


def test_plummer_profile():
    a = 3 * np.pi / 16
    Mp = 1.0 / 0.98518534                              # truncation at 10a renormalised to M = 1
    for rm, arm, cnt, r, ar in _radial_profile("plummer", 1 << 14, 7, np.array([0.2, 0.35, 0.6, 1.0, 1.6, 2.5])):
        want = np.mean(-Mp * r / (r * r + a * a) ** 1.5)
        assert cnt > 500 and arm == pytest.approx(want, rel=0.03)


def test_hernquist_profile():
    Mp = (101.0 / 100.0) ** 2
    for rm, arm, cnt, r, ar in _radial_profile("hernquist", 1 << 16, 8, np.array([0.3, 0.6, 1.0, 2.0, 4.0, 8.0])):
        want = np.mean(-Mp / (r + 1.0) ** 2)
        assert cnt > 500 and arm == pytest.approx(want, rel=0.03)


def test_cold_sphere_profile():
    for rm, arm, cnt, r, ar in _radial_profile("cold_sphere", 1 << 14, 9, np.array([0.3, 0.5, 0.7, 0.85, 0.97])):
        assert cnt > 500 and arm == pytest.approx(np.mean(-r), rel=0.03)
