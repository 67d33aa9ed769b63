"""Sink-sharded stepping over several replicas (PAPER.md:113-122 without the LET).

Every rank holds ALL particles and builds the same tree (the build is a small part of a cycle); the
sinks are divided: rank r evaluates the sink groups whose first particle lies in its range of store
slots (hyb_set_sink_range) and writes zeros elsewhere, one all-reduce(SUM) of the 16-byte accelerations
after each force evaluation puts the full result on every rank (x + 0 = x exactly, so the result does not
depend on the number of ranks), and every rank then applies the same kick / drift to all particles, so the
replicas stay bit-identical and no positions are ever exchanged.  The cycle is hyb_step's (R21),
issued call by call so that the exchange sits between the force evaluation and the kick.

This module holds no arithmetic of the method: `engine` is anything with the Hyb call names (the CUDA
binding; the CPU tests drive the same code over gloo with a stand-in of their own).  Unmeasured on
hardware: the pool offers one GPU per box (BASELINE.json's north_star keeps the headline on one GPU)."""
from __future__ import annotations

import numpy as np


def sink_ranges(n: int, world: int, cost: np.ndarray | None = None):
    """Boundaries b[0] = 0 <= ... <= b[world] = n of contiguous store-slot ranges, one per rank.
    cost (optional, length n, >= 0): per-sink work estimate, e.g. the list length of the sink's group at the
    previous evaluation; the ranges then carry about equal cost (the paper balances N_local + N_hard the same
    way).  Deterministic: every rank computes the same boundaries from the same input."""
    if cost is None:
        return [(n * r) // world for r in range(world + 1)]
    c = np.asarray(cost, dtype=np.float64)
    assert c.shape == (n,) and np.all(c >= 0)
    cum = np.concatenate(([0.0], np.cumsum(c)))
    if cum[-1] <= 0:
        return [(n * r) // world for r in range(world + 1)]
    b = [0]
    for r in range(1, world):
        b.append(int(np.searchsorted(cum, cum[-1] * r / world, side="left")))
    b.append(n)
    for r in range(1, world + 1):                   # monotone, whatever the rounding did
        b[r] = max(b[r], b[r - 1])
    return b


class ShardedHyb:
    """R21 cycles with the force evaluations divided over the ranks of a torch.distributed group."""

    def __init__(self, engine, params, rank: int, world: int, all_reduce, bounds=None):
        """engine: Hyb-like (build_tree, build_tree_hard, soft_force, hard_force, kick_drift, set_sink_range,
        a_soft, a_hard tensors, n).  all_reduce(tensor): in-place element-wise sum over the ranks."""
        self.e, self.p, self.rank, self.world, self.all_reduce = engine, params, rank, world, all_reduce
        self.bounds = bounds if bounds is not None else sink_ranges(engine.n, world)
        self.acc_valid = False
        self._apply_range()

    def _apply_range(self):
        self.e.set_sink_range(self.bounds[self.rank], self.bounds[self.rank + 1])

    def rebalance(self, cost_local):
        """cost_local: per-sink cost known to this rank (zeros for sinks it did not evaluate), torch tensor of
        length n; summed over the ranks, then every rank derives the same new ranges."""
        self.all_reduce(cost_local)
        self.bounds = sink_ranges(self.e.n, self.world, cost_local.detach().cpu().numpy())
        self._apply_range()
        self.acc_valid = False

    def _soft(self):
        self.e.build_tree()
        self.e.soft_force()
        self.all_reduce(self.e.a_soft)
        self.all_reduce(self.e.a_hard)

    def _hard(self):
        self.e.build_tree_hard()
        self.e.hard_force()
        self.all_reduce(self.e.a_hard)

    def step(self, n_soft_steps: int = 1):
        p = self.p
        split, nsub = p.split != 0, p.n_sub
        dts = np.float32(p.dt_soft)
        dth = np.float32(dts / np.float32(nsub))
        half = np.float32(0.5)
        if not self.acc_valid:
            self._soft()
            self.acc_valid = True
        for _ in range(n_soft_steps):
            for k in range(nsub):
                # opening kick(s) + drift; inside a cycle the closing half kick of one substep and the opening
                # half kick of the next use the same acceleration and are one kick (as in hyb_step)
                open_c = float(half * dth) if k == 0 else float(dth)
                soft_step = (not split) or k == nsub - 1
                if split:
                    self.e.kick_drift(float(half * dts) if k == 0 else 0.0, open_c, float(dth))
                else:
                    self.e.kick_drift(open_c, 0.0, float(dth))
                if soft_step:
                    self._soft()
                else:
                    self._hard()
                if k == nsub - 1:
                    if split:
                        self.e.kick_drift(float(half * dts), float(half * dth), 0.0)
                    else:
                        self.e.kick_drift(float(half * dth), 0.0, 0.0)
