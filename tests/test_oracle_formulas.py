"""Pins for the oracle's closed-form pieces: K (Eq. 10), r_b (Eq. 5), keys (T2-T5), sort (T6)."""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if not ln.startswith("#") and ln.strip()]


def test_K_exact_rationals():
    # PAPER.md:82-85 Eq. 10 with Y = (R2 - r)/(R2 - R1): pick R1 = 1, R2 = 2 so r = 2 - Y.
    for yn, yd, kn, kd in _rows("k_eq10.txt"):
        Y = Fraction(int(yn), int(yd))
        r = 2.0 - float(Y)
        assert O.K(r, 1.0, 2.0) == pytest.approx(float(Fraction(int(kn), int(kd))), rel=1e-13, abs=1e-18)
    assert O.K(1.5, 1.0, 2.0) == 53.0 / 512.0          # the mid-zone value


def test_K_branches_and_monotone():
    assert O.K(0.5, 1.0, 2.0) == 1.0 and O.K(1.0, 1.0, 2.0) == 1.0       # Y >= 1
    assert O.K(2.0, 1.0, 2.0) == 0.0 and O.K(7.0, 1.0, 2.0) == 0.0       # Y <= 0
    r = np.linspace(1.0, 2.0, 2001)
    k = np.array([O.K(x, 1.0, 2.0) for x in r])
    assert np.all(np.diff(k) <= 1e-15)
    # dK/dY = 60 Y^5 (1 - Y^2)^2; dK/dr = -dK/dY for R2 - R1 = 1
    Y = 2.0 - r[1:-1]
    num = -(k[2:] - k[:-2]) / (r[2:] - r[:-2])
    assert np.allclose(num, 60 * Y ** 5 * (1 - Y ** 2) ** 2, atol=2e-5)


def test_K_scaling_invariance():
    # K depends on r only through Y
    for y in (0.1, 0.37, 0.9):
        assert O.K(0.03 - y * 0.027, 0.003, 0.03) == pytest.approx(O.K(2.0 - y, 1.0, 2.0), rel=1e-12)


def test_K_poly7_alternative():
    # north_star's K(x) = 1 - x^4 (35 - 84x + 70x^2 - 20x^3): x=1/2 -> 1/2, 1/4 -> 3807/4096, 3/4 -> 289/4096
    assert O.K(1.5, 1.0, 2.0, 1) == pytest.approx(0.5, rel=1e-14)
    assert O.K(1.25, 1.0, 2.0, 1) == pytest.approx(3807 / 4096, rel=1e-14)
    assert O.K(1.75, 1.0, 2.0, 1) == pytest.approx(289 / 4096, rel=1e-13)
    assert O.K(0.9, 1.0, 2.0, 1) == 1.0 and O.K(2.1, 1.0, 2.0, 1) == 0.0


def test_rb_worked_values():
    for b, B2, aerr, rb in _rows("rb_eq5.txt"):
        assert O.rb(float(b), float(B2), float(aerr)) == pytest.approx(float(rb), rel=1e-14, abs=1e-300)


def test_rb_is_root_of_salmon_warren_bound():
    # Eq. 5 is the positive root of r (r - b_max) = sqrt(3 B_2 / a_err)
    rng = np.random.default_rng(5)
    for _ in range(50):
        b, B2, aerr = rng.uniform(0, 3), rng.uniform(0, 5), 2.0 ** -rng.integers(1, 12)
        r = O.rb(b, B2, aerr)
        assert r >= b
        assert r * (r - b) == pytest.approx(np.sqrt(3 * B2 / aerr), rel=1e-12, abs=1e-12)


# ------------------------------------------------------------------ keys


def _params(**kw):
    d = dict(G=1.0, eps=0.01, theta=0.5, a_err=2.0 ** -8, r_in=0.01, r_out=0.1, dt_soft=0.01, n_sub=4,
             leaf_max=8, group_max=32, mac=0, kfunc=0, split=1, grouping=1, hard_tree=0)
    d.update(kw)
    return O.OrcParams(**d)


def _tree(xyz, **kw):
    xyz = np.asarray(xyz, dtype=np.float64)
    p = np.zeros((len(xyz), 4), np.float32)
    p[:, :3] = xyz
    p[:, 3] = 1.0 / len(xyz)
    return O.Tree(p, _params(**kw)), p


def test_keys_lattice_bits():
    # cube [0, 2^21]: inv = 1 exactly, so q = floor(x); unit steps set single bits (T5)
    top = float(2 ** 21)
    pts = [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (2, 0, 0), (0, 2, 0), (0, 0, 2), (3, 5, 6), (top, top, top)]
    t, _ = _tree(pts)
    k = t.get("keys")
    assert list(k[:7]) == [0, 4, 2, 1, 32, 16, 8]
    # (3,5,6): x=011 y=101 z=110 -> digits (bit2..0): b2: x0 y1 z1 = 3; b1: x1 y0 z1 = 5; b0: x1 y1 z0 = 6
    assert k[7] == (3 << 6) | (5 << 3) | 6
    assert k[8] == 2 ** 63 - 1                    # clamp at the maximal extent


def test_keys_against_second_quantiser():
    rng = np.random.default_rng(11)
    xyz = rng.normal(size=(64, 3)).astype(np.float32)
    t, p = _tree(xyz)
    keys = t.get("keys")
    lo = p[:, :3].min(axis=0); hi = p[:, :3].max(axis=0)
    L = max(Fraction(float(hi[a])) - Fraction(float(lo[a])) for a in range(3))
    assert float(L) == t.get("root_L")[0]
    # exact rational quantiser using the fp64 inv the spec prescribes (T3): inv = 2097152.0 / L
    inv = 2097152.0 / float(L)
    for i in range(64):
        key = 0
        q = []
        for a in range(3):
            d = float(p[i, a]) - float(lo[a])            # exact in fp64? the spec says fp64 subtract
            s = np.float64(d) * np.float64(inv)
            q.append(min(int(np.floor(s)), 2097151))
        for b in range(21):
            key |= ((q[0] >> b) & 1) << (3 * b + 2) | ((q[1] >> b) & 1) << (3 * b + 1) | ((q[2] >> b) & 1) << (3 * b)
        assert key == int(keys[i])
    # octant digit at level 0 is (x<<2 | y<<1 | z) of the top quantised bits
    mid = [float(lo[a]) + float(L) / 2 for a in range(3)]
    for i in range(64):
        dig = int(keys[i] >> 60) & 7
        exp = (int(p[i, 0] >= mid[0]) << 2) | (int(p[i, 1] >= mid[1]) << 1) | int(p[i, 2] >= mid[2])
        if all(abs(float(p[i, a]) - mid[a]) > 1e-5 for a in range(3)):
            assert dig == exp


def test_keys_degenerate_box():
    t, _ = _tree([(0.5, 0.5, 0.5)] * 5)
    assert t.get("root_L")[0] == 1.0 and np.all(t.get("keys") == 0)
    assert list(t.get("perm")) == [0, 1, 2, 3, 4]


# ------------------------------------------------------------------ sort


def test_sort_stable_equivalence(ic0, tree0):
    keys = tree0.get("keys"); perm = tree0.get("perm")
    assert np.array_equal(np.sort(perm), np.arange(len(perm)))
    assert np.array_equal(perm, np.argsort(keys, kind="stable"))
    assert np.array_equal(tree0.get("keys_sorted"), keys[perm])
    assert np.array_equal(tree0.get("pos_sorted"), ic0[0][perm])


def test_sort_many_duplicates():
    rng = np.random.default_rng(3)
    base = rng.uniform(size=(7, 3))
    xyz = np.concatenate([base[rng.integers(0, 7, 500)], [[0, 0, 0], [1, 1, 1]]])
    t, _ = _tree(xyz)
    keys = t.get("keys")
    assert len(np.unique(keys)) <= 9
    assert np.array_equal(t.get("perm"), np.argsort(keys, kind="stable"))
