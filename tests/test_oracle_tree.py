"""Pins for the oracle's octree (T7), moments (T8-T10), groups (T11) and lists (T12-T13)."""
import numpy as np
import pytest

from oracle import oracle as O
from test_oracle_formulas import _params, _tree

NOCHILD = 0xFFFFFFFF


def _arrays(t):
    return {k: t.get(k) for k in ("level", "first", "count", "child", "nchild", "parent", "level_offset")}


def check_octree_invariants(t, leaf_max):
    a = _arrays(t); ks = t.get("keys_sorted"); nn = t.nn
    lev, first, count, child, nchild, parent = (a[k] for k in ("level", "first", "count", "child", "nchild", "parent"))
    assert lev[0] == 0 and first[0] == 0 and count[0] == t.n and parent[0] == NOCHILD
    # BFS: levels non-decreasing, first ascending within a level, level_offset consistent
    assert np.all(np.diff(lev.astype(int)) >= 0)
    lo = a["level_offset"]
    for l in range(22):
        s, e = lo[l], lo[l + 1]
        assert np.all(lev[s:e] == l)
        assert np.all(np.diff(first[s:e].astype(np.int64)) > 0)
    assert lo[22] == nn
    internal = child != NOCHILD
    assert np.array_equal(internal, (count > leaf_max) & (lev < 21))
    leafsum = count[~internal].sum()
    assert leafsum == t.n
    nxt = 1
    for k in np.nonzero(internal)[0]:
        c0, nc = int(child[k]), int(nchild[k])
        assert c0 == nxt and 1 <= nc <= 8            # children contiguous, in BFS order
        nxt += nc
        assert np.all(parent[c0:c0 + nc] == k) and np.all(lev[c0:c0 + nc] == lev[k] + 1)
        assert first[c0] == first[k] and count[c0:c0 + nc].sum() == count[k]
        assert np.array_equal(first[c0 + 1:c0 + nc], first[c0:c0 + nc - 1] + count[c0:c0 + nc - 1])
        digs = [(int(ks[first[c]]) >> (60 - 3 * int(lev[k]))) & 7 for c in range(c0, c0 + nc)]
        assert digs == sorted(set(digs))               # digit order, one child per non-empty digit
    assert nxt == nn
    for k in range(nn):                                # keys of a node share the top 3*level bits
        sh = 63 - 3 * int(lev[k])
        seg = ks[first[k]:first[k] + count[k]]
        if sh < 63:
            assert len(np.unique(seg >> np.uint64(sh))) == 1


def test_octree_invariants_cfg0(tree0, cfg0):
    check_octree_invariants(tree0, cfg0.leaf_max)


@pytest.mark.parametrize("leaf_max", [1, 2, 8])
def test_octree_vs_geometric_bisection(leaf_max):
    """Independent pointer octree by recursive geometric bisection of the T3 cube."""
    rng = np.random.default_rng(leaf_max)
    xyz = np.concatenate([rng.uniform(size=(200, 3)) ** 2, [[0, 0, 0], [1, 1, 1]]]).astype(np.float32)
    xyz[-1] = 1.0                                        # cube = [0,1]^3, inv = 2^21 exactly
    t, p = _tree(xyz, leaf_max=leaf_max, group_max=max(leaf_max, 32))
    ps = t.get("pos_sorted")[:, :3].astype(np.float64)
    want = set()

    def rec(idx, lo, size, level):
        want.add((level, int(idx.min()), len(idx)))
        if len(idx) <= leaf_max or level == 21:
            return
        half = size / 2
        for o in range(8):
            sel = idx
            for a, bit in zip(range(3), (4, 2, 1)):
                x = np.minimum(ps[sel, a], np.nextafter(1.0, 0.0))     # clamp at the top face (T4)
                m = (x >= lo[a] + half) if (o & bit) else (x < lo[a] + half)
                sel = sel[m]
            if len(sel):
                assert np.array_equal(sel, np.arange(sel.min(), sel.min() + len(sel)))   # contiguous in Morton order
                rec(sel, [lo[a] + (half if (o & bit) else 0.0) for a, bit in zip(range(3), (4, 2, 1))], half, level + 1)

    rec(np.arange(t.n), [0.0, 0.0, 0.0], 1.0, 0)
    a = _arrays(t)
    got = set(zip(a["level"].tolist(), a["first"].tolist(), a["count"].tolist()))
    assert got == want


def test_octree_depth_limit_and_coincident_points():
    xyz = np.concatenate([np.full((40, 3), 0.3), [[0, 0, 0], [1, 1, 1]]])
    t, _ = _tree(xyz, leaf_max=4, group_max=8)
    check_octree_invariants(t, 4)
    a = _arrays(t)
    deep = a["level"] == 21
    assert deep.any() and a["count"][deep].max() == 40 and np.all(a["child"][deep] == NOCHILD)
    gf, gc = t.get("gfirst"), t.get("gcount")
    assert gc.sum() == t.n and gc.max() <= 8
    assert np.array_equal(gf, np.concatenate([[0], np.cumsum(gc)[:-1]]))
    assert sorted(gc.tolist(), reverse=True)[:5] == [8, 8, 8, 8, 8]         # 40 = 5 chunks of 8


def test_moments_root_and_boxes(tree0, ic0):
    ps = tree0.get("pos_sorted").astype(np.float64)
    m, x = ps[:, 3], ps[:, :3]
    M64, C64, com_m = tree0.get("M64"), tree0.get("C64"), tree0.get("com_m")
    assert M64[0] == pytest.approx(m.sum(), rel=1e-12)
    com = (m[:, None] * x).sum(axis=0) / m.sum()
    assert np.allclose(C64[0], com, rtol=0, atol=1e-12)
    first, count, child = tree0.get("first"), tree0.get("count"), tree0.get("child")
    nlo, nhi = tree0.get("nlo"), tree0.get("nhi")
    for k in range(tree0.nn):
        seg = ps[first[k]:first[k] + count[k]]
        assert np.array_equal(nlo[k], seg[:, :3].min(axis=0).astype(np.float32))
        assert np.array_equal(nhi[k], seg[:, :3].max(axis=0).astype(np.float32))
        c = (seg[:, 3:4] * seg[:, :3]).sum(axis=0) / seg[:, 3].sum()
        assert np.allclose(C64[k], c, rtol=0, atol=1e-13)
        assert np.all(C64[k] >= nlo[k] - 1e-12) and np.all(C64[k] <= nhi[k] + 1e-12)
        assert np.array_equal(com_m[k, :3], C64[k].astype(np.float32)) and com_m[k, 3] == np.float32(M64[k])
        if count[k] == 1:
            assert np.array_equal(com_m[k, :3], seg[0, :3].astype(np.float32))      # bit-exact


def test_theta_mode_ropen(tree0, cfg0):
    L = np.float32(tree0.get("root_L")[0])
    lev = tree0.get("level").astype(np.int32)
    l = (L * np.float32(2.0) ** (-lev)).astype(np.float32)
    r = (l / np.float32(cfg0.theta)).astype(np.float32)
    assert np.array_equal(tree0.get("ropen2"), (r * r).astype(np.float32))
    t0 = O.Tree(tree0.get("pos_sorted"), O.params_from(cfg0, theta=0.0))
    assert np.all(np.isinf(t0.get("ropen2")))


def test_abs_mode_B2_bmax(cfg0, ic0):
    t = O.Tree(ic0[0], O.params_from(cfg0, mac=1))
    ps = t.get("pos_sorted").astype(np.float64)
    first, count = t.get("first"), t.get("count")
    C64, B2, bmax, ropen2 = t.get("C64"), t.get("B2"), t.get("bmax"), t.get("ropen2")
    nlo, nhi = t.get("nlo").astype(np.float64), t.get("nhi").astype(np.float64)
    for k in list(range(0, 60)) + list(range(60, t.nn, 37)):
        seg = ps[first[k]:first[k] + count[k]]
        d2 = ((seg[:, :3] - C64[k]) ** 2).sum(axis=1)
        assert B2[k] == pytest.approx((seg[:, 3] * d2).sum(), rel=1e-10, abs=1e-22)     # Eq. 6 directly
        assert bmax[k] == pytest.approx(np.sqrt(d2.max()), rel=1e-14)                 # R9: exact maximum
        centre = 0.5 * (nlo[k] + nhi[k])
        assert bmax[k] <= 0.5 * np.linalg.norm(nhi[k] - nlo[k]) + np.linalg.norm(C64[k] - centre) + 1e-12
        rb = np.float32(O.rb(bmax[k], B2[k], float(np.float32(cfg0.a_err))))
        assert ropen2[k] == rb * rb
    single = np.nonzero(count == 1)[0]
    assert len(single) and np.all(ropen2[single] == 0.0)                               # single particle -> r_b = 0


def _groups_tile(t, group_max):
    gf, gc = t.get("gfirst").astype(np.int64), t.get("gcount").astype(np.int64)
    assert gf[0] == 0 and np.array_equal(gf[1:], np.cumsum(gc)[:-1]) and gc.sum() == t.n
    assert gc.max() <= group_max and gc.min() >= 1
    return gf, gc


def test_groups_single_nodes(cfg0, ic0):
    """grouping 0 (R17, first reading): a group is a maximal tree node of <= group_max particles"""
    t = O.Tree(ic0[0], O.params_from(cfg0, grouping=0))
    gf, gc = _groups_tile(t, cfg0.group_max)
    first, count, parent = t.get("first"), t.get("count"), t.get("parent")
    for f, c in zip(gf, gc):
        # several nodes on a one-child chain can share (first,count); any of them works for the parent check
        ks = [k for k in range(t.nn) if first[k] == f and count[k] == c]
        assert ks, "every group is a tree node here (no level-21 chunks in cfg0)"
        top = min(ks)
        assert top == 0 or count[parent[top]] > cfg0.group_max


def test_groups(tree0, cfg0):
    """grouping 1 (the configs' default): greedy runs of consecutive small children of one cell"""
    assert cfg0.grouping in (1, 2) and tree0.params.grouping == 1
    gf, gc = _groups_tile(tree0, cfg0.group_max)
    gm = cfg0.group_max
    first, count, parent, child, nchild = (tree0.get(k).astype(np.int64) for k in ("first", "count", "parent", "child", "nchild"))
    # brute force, written differently from the oracle: walk the cells that are too big for one group
    # and cut their list of children wherever the running total would pass group_max
    starts = set()
    big = [k for k in range(tree0.nn) if count[k] > gm]
    for k in big:
        assert child[k] != NOCHILD, "no level-21 chunks in cfg0"
        kids = list(range(child[k], child[k] + nchild[k]))
        i = 0
        while i < len(kids):
            if count[kids[i]] > gm:
                i += 1
                continue
            j, tot = i, 0
            while j < len(kids) and count[kids[j]] <= gm and tot + count[kids[j]] <= gm:
                tot += count[kids[j]]; j += 1
            starts.add(int(first[kids[i]]))
            i = j
    assert starts == set(int(f) for f in gf)
    # fewer and fuller groups than one node per group, and never across the parent cell
    t0 = O.Tree(tree0.get("pos_sorted"), O.params_from(cfg0, grouping=0))
    assert tree0.ng < t0.ng and set(int(f) for f in gf) <= set(int(f) for f in t0.get("gfirst"))
    ps = tree0.get("pos_sorted")
    glo, ghi = tree0.get("glo"), tree0.get("ghi")
    for g in range(0, tree0.ng, 17):
        seg = ps[gf[g]:gf[g] + gc[g], :3]
        assert np.array_equal(glo[g], seg.min(axis=0)) and np.array_equal(ghi[g], seg.max(axis=0))


def test_lists_completeness_and_modes(tree0, cfg0):
    count = tree0.get("count").astype(np.int64)
    nc, npart, nh = tree0.walk_counts(O.MODE_HYBRID)
    nc_h, np_h, nh_h = tree0.walk_counts(O.MODE_HARD)
    nc_n, np_n, nh_n = tree0.walk_counts(O.MODE_NORMAL)
    assert np.array_equal(nh, nh_h) and np.all(nc_h == 0) and np.array_equal(np_h, nh_h)
    assert np.all(nh <= npart) and np.all(nh_n == 0)
    assert np.all(np_n <= npart) and np.all(nc_n.astype(int) + np_n >= 1)
    for mode in (O.MODE_HYBRID, O.MODE_NORMAL):
        for g in range(0, tree0.ng, 13):
            cells, parts, hard = tree0.walk_lists(mode, g)
            assert count[cells].sum() + len(parts) == tree0.n                  # every particle exactly once
            covered = np.zeros(tree0.n, np.int32)
            first = tree0.get("first")
            for c in cells:
                covered[first[c]:first[c] + count[c]] += 1
            covered[parts] += 1
            assert np.all(covered == 1)


def test_lists_theta0_opens_everything(cfg0, ic0):
    t = O.Tree(ic0[0], O.params_from(cfg0, theta=0.0))
    nc, npart, nh = t.walk_counts(O.MODE_HYBRID)
    assert np.all(nc == 0) and np.all(npart == t.n)


def test_hard_list_contains_all_neighbours(tree0, cfg0):
    ps = tree0.get("pos_sorted")[:, :3].astype(np.float64)
    gf, gc = tree0.get("gfirst"), tree0.get("gcount")
    for g in range(0, tree0.ng, 7):
        _, parts, hard = tree0.walk_lists(O.MODE_HARD, g)
        _, parts2, hard2 = tree0.walk_lists(O.MODE_HYBRID, g)
        assert hard.all() and set(parts.tolist()) == set(parts2[hard2].tolist())
        mem = ps[gf[g]:gf[g] + gc[g]]
        d = np.sqrt(((ps[None, :, :] - mem[:, None, :]) ** 2).sum(axis=2)).min(axis=0)
        need = set(np.nonzero(d < cfg0.r_out)[0].tolist())
        assert need <= set(parts.tolist())
