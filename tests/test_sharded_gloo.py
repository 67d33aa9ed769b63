"""world_size-2 gloo test (CPU) of the sink-sharded cycle (paper_1406_6158_b200/sharded.py):
the partition of the sinks, the exchange after every force evaluation and the order of the calls of a cycle.
The force evaluations come from an oracle-backed stand-in with the call names of the CUDA binding, restricted
to the sink groups of the rank's range exactly as hyb_set_sink_range restricts the kernels; two ranks must
reproduce the single-rank run bit for bit (every sink is evaluated by exactly one rank and x + 0 = x)."""
import os
import socket
from types import SimpleNamespace

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1406_6158_b200.sharded import ShardedHyb, sink_ranges


class OracleEngine:
    """the Hyb call names on top of the oracle (float32 store in Morton order, like the CUDA path)"""

    def __init__(self, cfg, pos, vel):
        from oracle import oracle as O
        self.O, self.cfg, self.n = O, cfg, pos.shape[0]
        self.pos, self.vel = pos.copy(), vel.copy()
        self.a_soft = torch.zeros(self.n, 4); self.a_hard = torch.zeros(self.n, 4)
        self.lo, self.hi = 0, self.n
        self.tree = None
        self.calls = []

    def set_sink_range(self, first, last):
        self.lo, self.hi = first, last

    def _build(self, **over):
        t = self.O.Tree(self.pos, self.O.params_from(self.cfg, **over))
        perm = t.get("perm")
        self.pos, self.vel = self.pos[perm], self.vel[perm]
        self.tree = t

    def build_tree(self):
        self.calls.append("build"); self._build()

    def build_tree_hard(self):
        self.calls.append("build_hard"); self._build(group_max=max(self.cfg.group_max // 2, self.cfg.leaf_max))

    def _mine(self):
        gf = self.tree.get("gfirst").astype(np.int64)
        return np.nonzero((gf >= self.lo) & (gf < self.hi))[0].astype(np.int64)

    def _store(self, dst, a):
        dst.zero_()
        dst[:, :3] = torch.from_numpy(a.astype(np.float32))

    def soft_force(self):
        self.calls.append("soft")
        g = self._mine()
        a_s, a_h, _ = self.tree.forces(self.O.MODE_HYBRID, g) if len(g) else (np.zeros((self.n, 3)),) * 2 + (None,)
        self._store(self.a_soft, a_s); self._store(self.a_hard, a_h)

    def hard_force(self):
        self.calls.append("hard")
        g = self._mine()
        _, a_h, _ = self.tree.forces(self.O.MODE_HARD, g) if len(g) else (None, np.zeros((self.n, 3)), None)
        self._store(self.a_hard, a_h)

    def kick_drift(self, c_soft, c_hard, dt):
        self.calls.append(("kick", c_soft != 0.0, c_hard != 0.0, dt != 0.0))
        f = np.float32
        self.vel[:, :3] += f(c_soft) * self.a_soft.numpy()[:, :3] + f(c_hard) * self.a_hard.numpy()[:, :3]
        self.pos[:, :3] += f(dt) * self.vel[:, :3]


def _run(rank, world, cycles=2, rebalance=False):
    from workloads import CONFIGS, make_ic
    cfg = CONFIGS[0].with_(n=1500, n_sub=3)
    pos, vel = make_ic(cfg.kind, cfg.n, 11)
    eng = OracleEngine(cfg, pos, vel)
    ar = (lambda t: dist.all_reduce(t)) if world > 1 else (lambda t: None)
    sh = ShardedHyb(eng, SimpleNamespace(split=cfg.split, n_sub=cfg.n_sub, dt_soft=cfg.dt_soft), rank, world, ar)
    sh.step(1)
    if rebalance:                       # per-sink cost = list length of the sink's group (zeros outside the range)
        nc, npart, nh = eng.tree.walk_counts(eng.O.MODE_HYBRID)
        gf, gc = eng.tree.get("gfirst"), eng.tree.get("gcount")
        cost = torch.zeros(cfg.n, dtype=torch.float64)
        for g in eng._mine():
            cost[gf[g]:gf[g] + gc[g]] = float(nc[g] + npart[g])
        sh.rebalance(cost)
    sh.step(cycles - 1)
    return eng, sh


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, out, rebalance):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    eng, sh = _run(rank, world, rebalance=rebalance)
    out.put((rank, eng.pos.copy(), eng.vel.copy(), eng.a_soft.numpy().copy(), eng.a_hard.numpy().copy(), list(sh.bounds),
             eng.calls))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("rebalance", [False, True])
def test_two_ranks_reproduce_one_rank(rebalance):
    ref, _ = _run(0, 1)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q, rebalance)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted((q.get(timeout=300) for _ in ps), key=lambda r: r[0])
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    for rank, pos, vel, a_s, a_h, bounds, calls in res:
        assert np.array_equal(pos, ref.pos) and np.array_equal(vel, ref.vel)            # replicas stay identical
        assert np.array_equal(a_s, ref.a_soft.numpy()) and np.array_equal(a_h, ref.a_hard.numpy())
        assert bounds[0] == 0 and bounds[-1] == 1500 and bounds == res[0][5]
        assert calls == ref.calls or rebalance
    if rebalance:
        assert res[0][5][1] != 750                    # the cost-balanced cut is not the equal-count cut


def test_cycle_is_the_r21_sequence():
    """one soft-step + (n - 1) hard-steps per cycle, the tree rebuilt before every evaluation"""
    eng, _ = _run(0, 1, cycles=1)
    assert eng.calls == ["build", "soft",
                         ("kick", True, True, True), "build_hard", "hard",
                         ("kick", False, True, True), "build_hard", "hard",
                         ("kick", False, True, True), "build", "soft",
                         ("kick", True, True, False)]


def test_sink_ranges():
    assert sink_ranges(10, 3) == [0, 3, 6, 10]
    assert sink_ranges(5, 1) == [0, 5]
    c = np.zeros(100); c[:10] = 9.0; c[10:] = 1.0            # 90 + 90: the heavy tenth is half of the work
    assert sink_ranges(100, 2, c) == [0, 10, 100]
    b = sink_ranges(1000, 7, np.random.default_rng(0).uniform(0, 1, 1000))
    assert b[0] == 0 and b[-1] == 1000 and all(x <= y for x, y in zip(b, b[1:]))
    assert sink_ranges(8, 4, np.zeros(8)) == [0, 2, 4, 6, 8]
