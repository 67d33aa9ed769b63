"""Seeded initial-condition samplers (NumPy, fp64 maths, cast to fp32 once).

Recipes:
  * Plummer sphere in Henon units, Aarseth-Henon-Wielen rejection for the speeds
    (the paper's own test model).
  * Hernquist sphere, isotropic speeds by rejection from the analytic distribution function.
  * cold uniform ball.
  * two-Plummer merger.
All draws come from numpy.random.Generator(PCG64(seed)) in a fixed block order, so an
(N, seed) pair always gives the same arrays.  Nothing here knows about trees or forces.
"""
from __future__ import annotations

import numpy as np

_PLUMMER_A = 3.0 * np.pi / 16.0


def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    """n unit vectors uniform on the sphere (z uniform in [-1,1], phi uniform)."""
    z = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def _fill_by_rejection(rng, n, draw):
    """Call draw(rng, m) -> accepted values (1-D) until n are collected; keeps draw order."""
    out = np.empty(n, dtype=np.float64)
    have = 0
    while have < n:
        m = max(1024, int(1.3 * (n - have)) + 16)
        acc = draw(rng, m)
        k = min(len(acc), n - have)
        out[have:have + k] = acc[:k]
        have += k
    return out


def _plummer_radii(rng, n, a, rmax):
    def draw(rng, m):
        x = rng.uniform(0.0, 1.0, m)
        x = x[x > 0.0]
        r = a / np.sqrt(x ** (-2.0 / 3.0) - 1.0)
        return r[r <= rmax]
    return _fill_by_rejection(rng, n, draw)


def _ahw_q(rng, n):
    """q = v / v_esc with density g(q) = q^2 (1-q^2)^(7/2), rejection against 0.1."""
    def draw(rng, m):
        q = rng.uniform(0.0, 1.0, m)
        y = rng.uniform(0.0, 0.1, m)
        return q[y < q * q * (1.0 - q * q) ** 3.5]
    return _fill_by_rejection(rng, n, draw)


def _recentre(pos, vel, mass):
    mt = mass.sum()
    pos -= (mass[:, None] * pos).sum(axis=0) / mt
    vel -= (mass[:, None] * vel).sum(axis=0) / mt


def _plummer64(rng, n, total_mass=1.0):
    a = _PLUMMER_A
    r = _plummer_radii(rng, n, a, 10.0 * a)
    pos = r[:, None] * _isotropic(rng, n)
    vesc = np.sqrt(2.0 * total_mass) * (r * r + a * a) ** (-0.25)
    q = _ahw_q(rng, n)
    vel = (q * vesc)[:, None] * _isotropic(rng, n)
    mass = np.full(n, total_mass / n)
    _recentre(pos, vel, mass)
    return pos, vel, mass


def plummer(n: int, seed: int):
    """Plummer sphere, G=M=1, a=3pi/16, radii truncated at 10a (BASELINE.json configs 0, 1)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return _pack(*_plummer64(rng, n))


def hernquist_df(E):
    """Hernquist (1990) isotropic distribution function f(E), G=M=a=1, E<0 the binding energy
    per unit mass (E = Phi + v^2/2).  Used only by the sampler and its unit test."""
    q2 = np.clip(-E, 0.0, 1.0)
    q = np.sqrt(q2)
    om = np.maximum(1.0 - q2, 1e-300)
    br = 3.0 * np.arcsin(q) + q * np.sqrt(om) * (1.0 - 2.0 * q2) * (8.0 * q2 * q2 - 8.0 * q2 - 3.0)
    return br / (8.0 * np.sqrt(2.0) * np.pi ** 3 * om ** 2.5)


def hernquist(n: int, seed: int):
    """Hernquist sphere rho ~ 1/(r (r+a)^3), a=M=G=1, truncated at 100a (BASELINE.json config 2)."""
    rng = np.random.Generator(np.random.PCG64(seed))

    def draw_r(rng, m):
        s = np.sqrt(rng.uniform(0.0, 1.0, m))
        s = s[s < 1.0]
        r = s / (1.0 - s)
        return r[r <= 100.0]
    r = _fill_by_rejection(rng, n, draw_r)
    pos = r[:, None] * _isotropic(rng, n)
    phi = -1.0 / (r + 1.0)
    vmax = np.sqrt(-2.0 * phi)
    # envelope of v^2 f(Phi+v^2/2) over v in [0, vmax]: tabulated on 8192 potentials psi=-Phi in
    # (0,1] (max over a 256-point grid in v), looked up as 1.1 x the larger neighbouring entry
    npsi = 8192
    psi_t = (np.arange(npsi + 1) + 0.5) / (npsi + 1)
    grid = (np.arange(256) + 0.5) / 256.0
    vg = grid[None, :] * np.sqrt(2.0 * psi_t)[:, None]
    tab = (vg * vg * hernquist_df(-psi_t[:, None] + 0.5 * vg * vg)).max(axis=1)
    k = np.clip(np.floor(-phi * (npsi + 1) - 0.5).astype(np.int64), 0, npsi - 1)
    env = 1.1 * np.maximum(tab[k], tab[k + 1])
    v = np.empty(n)
    todo = np.arange(n)
    while len(todo):
        u = rng.uniform(0.0, 1.0, len(todo)) * vmax[todo]
        y = rng.uniform(0.0, 1.0, len(todo)) * env[todo]
        ok = y < u * u * hernquist_df(phi[todo] + 0.5 * u * u)
        v[todo[ok]] = u[ok]
        todo = todo[~ok]
    vel = v[:, None] * _isotropic(rng, n)
    mass = np.full(n, 1.0 / n)
    _recentre(pos, vel, mass)
    return _pack(pos, vel, mass)


def cold_sphere(n: int, seed: int):
    """Cold uniform ball, R=1, M=1, zero velocities (BASELINE.json config 3)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    r = rng.uniform(0.0, 1.0, n) ** (1.0 / 3.0)
    pos = r[:, None] * _isotropic(rng, n)
    vel = np.zeros((n, 3))
    mass = np.full(n, 1.0 / n)
    _recentre(pos, vel, mass)
    return _pack(pos, vel, mass)


def two_plummer(n: int, seed: int):
    """Two Henon-unit Plummer spheres of n/2 particles each (each M=1, recentred), centred at
    x=-/+2 with y-velocities +/-0.3; total M=2 (BASELINE.json config 4)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    h = n // 2
    pa, va, ma = _plummer64(rng, h)
    pb, vb, mb = _plummer64(rng, n - h)
    pa[:, 0] -= 2.0
    pb[:, 0] += 2.0
    va[:, 1] += 0.3
    vb[:, 1] -= 0.3
    return _pack(np.concatenate([pa, pb]), np.concatenate([va, vb]), np.concatenate([ma, mb]))


def _pack(pos, vel, mass):
    """-> pos_m float32 [N,4] (x,y,z,m), vel float32 [N,4] (vx,vy,vz,0); the fp32 cast is the
    single point where inputs become what both the CUDA path and the oracle see."""
    n = len(mass)
    pm = np.zeros((n, 4), dtype=np.float32)
    pm[:, :3] = pos
    pm[:, 3] = mass
    vv = np.zeros((n, 4), dtype=np.float32)
    vv[:, :3] = vel
    return pm, vv


_GENERATORS = {"plummer": plummer, "hernquist": hernquist, "cold_sphere": cold_sphere,
               "two_plummer": two_plummer}


def make_ic(kind: str, n: int, seed: int):
    return _GENERATORS[kind](n, seed)
