"""The five BASELINE.json configurations (+ the paper's own parameter recipe)."""
from __future__ import annotations

from dataclasses import dataclass, replace


@dataclass(frozen=True)
class Config:
    name: str
    kind: str            # generator in workloads.ic
    n: int
    seed: int
    eps: float
    theta: float
    leaf_max: int
    group_max: int
    r_in: float
    r_out: float
    dt_soft: float
    n_sub: int
    n_soft_steps: int
    G: float = 1.0
    a_err: float = 2.0 ** -8     # PAPER.md:174 "typically a_err = 2^-8"
    mac: int = 0                 # 0 = theta, 1 = absolute MAC (Eq. 5-6)
    kfunc: int = 0               # 0 = paper Eq. 10
    split: int = 1               # 1 = hybrid, 0 = normal tree
    grouping: int = 2            # sink groups: 1 = runs of consecutive small sibling cells, 0 = single tree nodes,
                                 # 2 = 1, with runs of at most group_max / 2 for the trees of hyb_step that only a hard walk uses

    hard_tree: int = 0           # 0 = hard force by direct K-weighted sum (R20), 1 = the paper's MAC-approximated hard walk

    hard_refit: int = 0          # 0 = tree rebuilt before every force evaluation (paper), 1 = hard-only substeps refit the boxes

    hard_cut: int = 1            # T13 hard list: 0 = every particle of a leaf within r_out of the group box,
                                 # 1 = only the particles that are themselves within r_out of the group box (R30)

    def with_(self, **kw) -> "Config":
        return replace(self, **kw)


CONFIGS = [
    Config("cfg0_plummer_4k", "plummer", 1 << 12, 0, 0.01, 0.5, 8, 32, 0.01, 0.1, 1.0 / 128, 4, 64),
    Config("cfg1_plummer_128k", "plummer", 1 << 17, 1, 0.005, 0.5, 16, 64, 0.005, 0.05, 1.0 / 256, 4, 16),
    Config("cfg2_hernquist_1m", "hernquist", 1 << 20, 2, 0.002, 0.5, 16, 64, 0.003, 0.03, 1.0 / 512, 8, 8),
    Config("cfg3_cold_4m", "cold_sphere", 1 << 22, 3, 0.001, 0.6, 16, 64, 0.001, 0.01, 1.0 / 1024, 4, 4),
    Config("cfg4_merger_16m", "two_plummer", 1 << 24, 4, 0.0005, 0.5, 16, 64, 0.001, 0.01, 1.0 / 1024, 4, 2),
]
CFG4_THETAS = (0.3, 0.5, 0.75)
CFG4_ROUTS = (0.005, 0.01, 0.02)      # r_in = 0.1 r_out


def get_config(i: int) -> Config:
    return CONFIGS[i]


def paper_params(n: int, seed: int = 0) -> Config:
    """Plummer, eps = 0.1 N^-0.26, dt_h = eps/0.65, n = 4,
    R1 = 1.03 N^-1/3, R2 = 2 R1, absolute MAC with a_err = 2^-8."""
    eps = 0.1 * n ** -0.26
    r1 = 1.03 * n ** (-1.0 / 3.0)
    return Config(f"paper_plummer_{n}", "plummer", n, seed, eps, 0.5, 16, 64, r1, 2.0 * r1,
                  4 * eps / 0.65, 4, 1, mac=1)
