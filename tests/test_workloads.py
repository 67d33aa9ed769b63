"""Sanity of the seeded input generators (they hold none of the method's arithmetic)."""
import numpy as np
import pytest

from workloads import CONFIGS, make_ic, paper_params
from workloads.ic import hernquist_df


def test_deterministic_and_shapes():
    for kind in ("plummer", "hernquist", "cold_sphere", "two_plummer"):
        p, v = make_ic(kind, 2048, 5)
        p2, v2 = make_ic(kind, 2048, 5)
        assert p.dtype == np.float32 and p.shape == (2048, 4) and v.shape == (2048, 4)
        assert np.array_equal(p, p2) and np.array_equal(v, v2)
        assert np.all(np.isfinite(p)) and np.all(p[:, 3] > 0) and np.all(v[:, 3] == 0)
        p3, _ = make_ic(kind, 2048, 6)
        assert not np.array_equal(p, p3)


def test_plummer_henon_units():
    p, v = make_ic("plummer", 1 << 15, 0)
    m = p[:, 3].astype(np.float64)
    assert m.sum() == pytest.approx(1.0, rel=1e-6)
    r = np.linalg.norm(p[:, :3].astype(np.float64), axis=1)
    a = 3 * np.pi / 16
    assert r.max() <= 10 * a * 1.01
    assert np.median(r) == pytest.approx(a / np.sqrt(0.98518534 ** (-2 / 3) * 2 ** (2 / 3) - 1), rel=0.03)
    ke = 0.5 * (m * (v[:, :3].astype(np.float64) ** 2).sum(axis=1)).sum()
    assert ke == pytest.approx(0.25, rel=0.05)          # virial: T = -E = 1/4


def test_hernquist_df_reproduces_density():
    # with prefactor 1/(8 sqrt2 pi^3), int 4 pi v^2 f dv = rho = 1/(2 pi r (1+r)^3)
    for r in (0.1, 1.0, 5.0):
        phi = -1.0 / (1.0 + r)
        vmax = np.sqrt(-2 * phi)
        # substitution v = vmax sin(t) tames the integrable edge behaviour
        t = (np.arange(200000) + 0.5) / 200000 * (np.pi / 2)
        vv = vmax * np.sin(t)
        integrand = 4 * np.pi * vv ** 2 * hernquist_df(phi + 0.5 * vv ** 2) * vmax * np.cos(t)
        rho = integrand.sum() * (np.pi / 2) / 200000
        assert rho == pytest.approx(1.0 / (2 * np.pi * r * (1 + r) ** 3), rel=1e-6)


def test_two_plummer_layout():
    p, v = make_ic("two_plummer", 4096, 4)
    assert p[:2048, 0].mean() == pytest.approx(-2.0, abs=1e-5) and p[2048:, 0].mean() == pytest.approx(2.0, abs=1e-5)
    assert v[:2048, 1].mean() == pytest.approx(0.3, abs=1e-5) and v[2048:, 1].mean() == pytest.approx(-0.3, abs=1e-5)
    assert p[:, 3].astype(np.float64).sum() == pytest.approx(2.0, rel=1e-6)


def test_config_table_matches_baseline():
    ns = [c.n for c in CONFIGS]
    assert ns == [1 << 12, 1 << 17, 1 << 20, 1 << 22, 1 << 24]
    assert [c.n_sub for c in CONFIGS] == [4, 4, 8, 4, 4]
    assert CONFIGS[2].kind == "hernquist" and CONFIGS[2].r_out == 0.03 and CONFIGS[2].eps == 0.002
    pp = paper_params(1 << 20)
    assert pp.eps == pytest.approx(0.00272, rel=2e-3) and pp.r_in == pytest.approx(0.01014, rel=2e-3)
