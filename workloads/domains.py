"""Virtual process domains for the LET-counting experiment.

The paper cuts space into P = Px x Py x Pz cuboids by a multi-section of SAMPLED particles
(sampling rate R_samp = 2^-8, slabs of equal sample counts along x, then y inside
every slab, then z).  This module only produces those boxes from seeded samples; it is an input
generator (it holds none of the tree / force arithmetic) and serves the CUDA path and the oracle alike.
The paper additionally rebalances the sampling rate per process by the measured load (Eq. 12-13); with a
single GPU there is no per-process load to measure, so the plain equal-count multi-section is used.
"""
from __future__ import annotations

import numpy as np


def _cuts(vals: np.ndarray, parts: int) -> np.ndarray:
    """parts - 1 cut positions that put about the same number of samples into each part"""
    s = np.sort(vals)
    idx = (np.arange(1, parts) * len(s)) // parts
    return 0.5 * (s[idx - 1] + s[idx]) if len(s) > parts else np.linspace(s.min(), s.max(), parts + 1)[1:-1]


def virtual_domains(pos: np.ndarray, px: int, py: int, pz: int, seed: int, r_samp: float = 2.0 ** -8) -> np.ndarray:
    """float32 [P, 6] boxes (lo xyz, hi xyz), half-open, outermost faces at -inf / +inf."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = pos.shape[0]
    m = max(int(n * r_samp), 8 * px * py * pz)
    smp = pos[rng.choice(n, size=min(m, n), replace=False), :3].astype(np.float64)
    boxes = []
    xc = np.concatenate(([-np.inf], _cuts(smp[:, 0], px), [np.inf]))
    for i in range(px):
        sx = smp[(smp[:, 0] >= xc[i]) & (smp[:, 0] < xc[i + 1])]
        yc = np.concatenate(([-np.inf], _cuts(sx[:, 1], py), [np.inf]))
        for j in range(py):
            sy = sx[(sx[:, 1] >= yc[j]) & (sx[:, 1] < yc[j + 1])]
            zc = np.concatenate(([-np.inf], _cuts(sy[:, 2], pz), [np.inf]))
            for k in range(pz):
                boxes.append([xc[i], yc[j], zc[k], xc[i + 1], yc[j + 1], zc[k + 1]])
    return np.asarray(boxes, dtype=np.float32)
