"""Pins for the oracle's integrator (T16 / R21): textbook leapfrog, circular binary, reversibility,
second order, and the (unpinned-by-the-paper) energy drift bound on config 0."""
import numpy as np
import pytest

from oracle import oracle as O
from test_oracle_formulas import _params
from test_oracle_forces import _numpy_direct


def _state(p, v):
    return p[:, :3].astype(np.float64).copy(), v[:, :3].astype(np.float64).copy(), p[:, 3].copy()


def test_normal_mode_n1_is_textbook_kdk():
    # PAPER.md:42-45 Eq. 3-4 in synchronised (kick-drift-kick) form, forces by the definition Eq. 1-2
    rng = np.random.default_rng(1)
    p = rng.normal(size=(48, 4)).astype(np.float32); p[:, 3] = 1.0 / 48
    v = (0.3 * rng.normal(size=(48, 4))).astype(np.float32)
    G, eps, dt = 1.0, 0.1, 0.01
    x, vv, m = _state(p, v)
    P = _params(G=G, eps=eps, theta=0.0, dt_soft=dt, n_sub=1, split=0)
    O.step(x, vv, m, P, ncycles=3)
    xr, vr, _ = _state(p, v)
    dt32 = float(np.float32(dt))

    def acc(xc):
        q = np.zeros((48, 4), np.float32); q[:, :3] = xc.astype(np.float32); q[:, 3] = m
        return _numpy_direct(q, G, eps)
    a = acc(xr)
    for _ in range(3):
        vr += 0.5 * dt32 * a; xr += dt32 * vr; a = acc(xr); vr += 0.5 * dt32 * a
    assert np.allclose(x, xr, rtol=0, atol=1e-13) and np.allclose(vv, vr, rtol=0, atol=1e-13)


def _binary(d=0.3, eps=0.05, m1=0.5, m2=0.5, G=1.0):
    w = np.sqrt(G * (m1 + m2) / (d * d + eps * eps) ** 1.5)       # softened circular binary
    x = np.array([[-d * m2 / (m1 + m2), 0, 0], [d * m1 / (m1 + m2), 0, 0]], np.float64)
    v = np.array([[0, -w * d * m2 / (m1 + m2), 0], [0, w * d * m1 / (m1 + m2), 0]], np.float64)
    return x, v, np.array([m1, m2], np.float32), w


@pytest.mark.parametrize("split", [0, 1])
def test_circular_binary_second_order(split):
    d, eps = 0.3, 0.05
    errs = []
    for nper in (256, 512):
        x, v, m, w = _binary(d, eps)
        T = 2 * np.pi / w
        # r_in < d < r_out: the pair sits in the changeover zone, so both a_hard and a_soft are non-zero
        P = _params(eps=eps, dt_soft=T / nper, n_sub=2, split=split, r_in=0.2, r_out=0.5)
        O.step(x, v, m, P, ncycles=nper)
        x0, _, _, _ = _binary(d, eps)
        # positions are rounded to fp32 for every force evaluation (the store is fp32): error floor ~1e-7
        errs.append(np.abs(x - x0).max())
        sep = np.linalg.norm(x[1] - x[0])
        assert sep == pytest.approx(d, rel=2e-3)
    assert errs[0] < 5e-3 and 3.0 < errs[0] / errs[1] < 5.0              # halve dt -> error / 4


def test_time_reversibility(cfg0):
    from workloads import make_ic
    p, v = make_ic("plummer", 256, 12)
    x, vv, m = _state(p, v)
    x0, v0 = x.copy(), vv.copy()
    P = O.params_from(cfg0)
    O.step(x, vv, m, P, ncycles=3)
    assert np.abs(x - x0).max() > 1e-3
    vv *= -1.0
    O.step(x, vv, m, P, ncycles=3)
    assert np.abs(x - x0).max() < 1e-10 and np.abs(vv + v0).max() < 1e-10


def test_hybrid_equals_normal_when_everything_is_hard_or_soft():
    # K == 0 everywhere (r_out tiny) with n_sub = 1: the hybrid cycle is the plain leapfrog
    from workloads import make_ic
    p, v = make_ic("plummer", 128, 3)
    xa, va, m = _state(p, v); xb, vb, _ = _state(p, v)
    O.step(xa, va, m, _params(theta=0.0, dt_soft=0.01, n_sub=1, split=1, r_in=1e-9, r_out=2e-9), ncycles=2)
    O.step(xb, vb, m, _params(theta=0.0, dt_soft=0.01, n_sub=1, split=0), ncycles=2)
    assert np.allclose(xa, xb, rtol=0, atol=1e-14) and np.allclose(va, vb, rtol=0, atol=1e-14)


def test_energy_drift_cfg0(cfg0, ic0):
    """|dE/E0| < 1e-3 over the config's 64 soft steps.  The paper states no bound:
    PARITY UNPINNED -- this is our own bound."""
    p, v = ic0
    x, vv, m = _state(p, v)
    P = O.params_from(cfg0)
    k0, w0 = O.energy(x, vv, m, cfg0.G, cfg0.eps)
    assert (k0 + w0) == pytest.approx(-0.25, rel=0.05)              # Henon units: E = -1/4
    a_s, a_h = O.step(x, vv, m, P, ncycles=0)
    worst = 0.0
    for _ in range(4):
        O.step(x, vv, m, P, ncycles=cfg0.n_soft_steps // 4, a_soft=a_s, a_hard=a_h)
        k, w = O.energy(x, vv, m, cfg0.G, cfg0.eps)
        worst = max(worst, abs((k + w - k0 - w0) / (k0 + w0)))
    assert worst < 1e-3
