"""Pins for the opening rule of the oracle's walks (T12 rule (a), T13) and for Eq. 14-15 in the LET
counts -- derived a second time, in another way, from what the paper fixes.

PAPER.md:66 "If r_b > r_ij ... we further visit ... else we add the force from the cell",
PAPER.md:107-109 Eq. 11 (the distance is the minimum over the sinks that share the walk; reading R18:
group box to the stored centre of mass), Eq. 14 (send a cell unless r_ib < r_b),
PAPER.md:152-156 Eq. 15 (hard LET: only what lies within R_2 + b_max).

The oracle walks the tree with a stack, node by node.  Here nothing is walked: for one sink group (or
one virtual domain) the predicates "open" and "inside" are evaluated for EVERY node at once as NumPy
float32 arrays (one rounding per operation, like T12), the property "every proper ancestor is open"
is propagated down the breadth-first numbering (a parent has a smaller index than its children), and
the lists are then DEFINED as sets:
    cell list     = { k : reached(k) and not open(k) }
    opened leaves = { k : reached(k) and open(k) and k is a leaf }
The oracle's lists must be exactly these sets.  The opening radius itself is recomputed from the level
array (theta mode: float32(L) 2^-level / theta) or from Eq. 5-6 written as direct sums over the node's
particles (absolute mode), not through the oracle's parallel-axis upsweep.

Mutation check (done when this file was written, and repeated by test_mutants_are_caught on every run):
the oracle source with glo and ghi swapped in dist2_box_com, and a second copy that measures the distance
to the centre of the node's tight box instead of its centre of mass, are compiled to a scratch library;
both fail the set comparison below on the same inputs the real oracle passes; so does a copy with the
domain faces swapped in the r_ib of orc_let_count (test_let_mutant_is_caught).
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from oracle import oracle as O
from workloads import CONFIGS, make_ic
from workloads.domains import virtual_domains

NOCHILD = 0xFFFFFFFF
F = np.float32


def _sq3(e):
    """(e_x^2 + e_y^2) + e_z^2 in float32, every operation rounded on its own"""
    xx = e[:, 0] * e[:, 0]; yy = e[:, 1] * e[:, 1]; zz = e[:, 2] * e[:, 2]
    return (xx + yy) + zz


def _point_box_d2(p, lo, hi):
    """squared distance from points p [k,3] to the box [lo, hi], float32"""
    e = np.maximum(F(0), np.maximum(lo[None, :] - p, p - hi[None, :])).astype(F)
    return _sq3(e)


def _box_box_d2(blo, bhi, lo, hi):
    e = np.maximum(F(0), np.maximum(blo - hi[None, :], lo[None, :] - bhi)).astype(F)
    return _sq3(e)


def _reached(parent, ok_to_descend):
    """reached[k] = every proper ancestor a of k has ok_to_descend[a]; parents precede children"""
    r = np.zeros(len(parent), bool)
    r[0] = True
    for k in range(1, len(parent)):
        r[k] = r[parent[k]] and ok_to_descend[parent[k]]
    return r


def _arrays(t):
    return {k: t.get(k) for k in ("level", "parent", "child", "count", "first", "com_m", "ropen2", "nlo", "nhi", "glo",
                                  "ghi", "gfirst", "gcount")}


def expected_lists(a, g, mode, r_out, in_cut=None):
    """the T12/T13 lists of group g as sets, from whole-array predicates; in_cut (hard_cut = 1, R30): the
    particles that are themselves within r_out of the group box, as a boolean array over all particles"""
    glo, ghi = a["glo"][g].astype(F), a["ghi"][g].astype(F)
    d2a = _point_box_d2(a["com_m"][:, :3].astype(F), glo, ghi)
    d2b = _box_box_d2(a["nlo"].astype(F), a["nhi"].astype(F), glo, ghi)
    rout2 = F(r_out) * F(r_out)
    mac_open = d2a < a["ropen2"]
    near = d2b < rout2
    if mode == O.MODE_NORMAL:
        opened, kept = mac_open, np.ones_like(near)
    elif mode == O.MODE_HYBRID:
        opened, kept = mac_open | near, np.ones_like(near)
    else:                                   # hard walk: a node farther than r_out is dropped, the rest is opened
        opened, kept = near, near
    leaf = a["child"] == NOCHILD
    reach = _reached(a["parent"].astype(np.int64), opened & ~leaf)
    cells = set(np.nonzero(reach & kept & ~opened)[0].tolist())
    leaves = np.nonzero(reach & opened & leaf)[0]
    parts, hard = set(), set()
    for k in leaves:
        rng = range(int(a["first"][k]), int(a["first"][k] + a["count"][k]))
        parts.update(rng)
        if mode != O.MODE_NORMAL and near[k]:
            hard.update(j for j in rng if in_cut is None or in_cut[j])
    return cells, parts, hard


def check_tree_lists(walk_lists, a, ng, r_out, step, ps=None):
    """ps: sorted positions when the oracle under test was built with hard_cut = 1"""
    bad = 0
    for mode in (O.MODE_HYBRID, O.MODE_NORMAL, O.MODE_HARD):
        for g in range(0, ng, step):
            cells, parts, hard = walk_lists(mode, g)
            in_cut = None
            if ps is not None:
                in_cut = _point_box_d2(ps[:, :3].astype(F), a["glo"][g].astype(F), a["ghi"][g].astype(F)) < F(r_out) * F(r_out)
            ec, ep, eh = expected_lists(a, g, mode, r_out, in_cut)
            got_hard = set(parts[hard].tolist())
            if mode == O.MODE_HARD:
                cells = cells[:0]           # the hard walk reports no cell list
                ec = set()
            if set(cells.tolist()) != ec or set(parts.tolist()) != ep or got_hard != eh:
                bad += 1
            assert len(cells) == len(set(cells.tolist())) and len(parts) == len(set(parts.tolist()))
    return bad


@pytest.mark.parametrize("mac,hard_cut", [(0, 0), (1, 0), (0, 1)])
def test_walk_lists_are_the_sets_the_rule_defines(mac, hard_cut):
    cfg = CONFIGS[0].with_(mac=mac, hard_cut=hard_cut)
    pos, _ = make_ic(cfg.kind, cfg.n, cfg.seed)
    t = O.Tree(pos, O.params_from(cfg))
    a = _arrays(t)
    assert check_tree_lists(t.walk_lists, a, t.ng, cfg.r_out, 5, t.get("pos_sorted") if hard_cut else None) == 0
    # the accepted cells really are far (rule (a)) and every ancestor of a list entry really was opened:
    # restated per entry, as PAPER.md:66 puts it
    glo, ghi = a["glo"], a["ghi"]
    for g in range(0, t.ng, 11):
        cells, parts, _ = t.walk_lists(O.MODE_NORMAL, g)
        d2a = _point_box_d2(a["com_m"][:, :3].astype(F), glo[g].astype(F), ghi[g].astype(F))
        assert np.all(d2a[cells] >= a["ropen2"][cells])
        anc = set()
        for k in cells.tolist():
            k = int(a["parent"][k])
            while k != NOCHILD and k not in anc:
                anc.add(k); k = int(a["parent"][k])
        anc = np.array(sorted(anc), np.int64)
        assert np.all(d2a[anc] < a["ropen2"][anc])


def test_opening_radius_theta_mode():
    """T10: r_open = float32(L) 2^-level / theta, from the level array (R27: geometric cell side)"""
    cfg = CONFIGS[0]
    pos, _ = make_ic(cfg.kind, cfg.n, cfg.seed)
    for theta in (0.5, 0.75, 0.3):
        t = O.Tree(pos, O.params_from(cfg, theta=theta))
        L = F(t.get("root_L")[0])
        side = np.ldexp(np.full(t.nn, L, F), -t.get("level").astype(np.int32)).astype(F)
        r = (side / F(theta)).astype(F)
        assert np.array_equal(t.get("ropen2"), (r * r).astype(F))
        # the side really is the side of the node's Morton cell: its particles fit inside one
        ext = (t.get("nhi") - t.get("nlo")).max(axis=1)
        assert np.all(ext <= side * F(1 + 1e-6))


def test_opening_radius_absolute_mode_from_direct_sums():
    """Eq. 5-6 with b_max and B_2 written as plain sums over the node's own particles
    about its own centre of mass (the oracle climbs the tree with the parallel-axis theorem instead)."""
    cfg = CONFIGS[0].with_(mac=1)
    pos, _ = make_ic(cfg.kind, cfg.n, cfg.seed)
    t = O.Tree(pos, O.params_from(cfg))
    ps = t.get("pos_sorted").astype(np.float64)
    first, count = t.get("first").astype(np.int64), t.get("count").astype(np.int64)
    rng = np.random.default_rng(4)
    for k in np.concatenate(([0, 1, 2], rng.choice(t.nn, 200, replace=False))):
        seg = ps[first[k]:first[k] + count[k]]
        M = seg[:, 3].sum()
        com = (seg[:, 3:4] * seg[:, :3]).sum(axis=0) / M
        d2 = ((seg[:, :3] - com) ** 2).sum(axis=1)
        bmax, B2 = np.sqrt(d2.max()), (seg[:, 3] * d2).sum()
        assert t.get("bmax")[k] == pytest.approx(bmax, rel=1e-9, abs=1e-15)
        assert t.get("B2")[k] == pytest.approx(B2, rel=1e-8, abs=1e-20)
        rb = bmax / 2 + np.sqrt(bmax * bmax / 4 + np.sqrt(3 * B2 / float(F(cfg.a_err))))
        assert np.sqrt(float(t.get("ropen2")[k])) == pytest.approx(rb, rel=1e-6)
        # Eq. 5 is the positive root of r (r - b_max) = sqrt(3 B_2 / a_err) (Salmon-Warren bound)
        assert rb * (rb - bmax) == pytest.approx(np.sqrt(3 * B2 / float(F(cfg.a_err))), rel=1e-9, abs=1e-15)


# ---------------------------------------------------------------- Eq. 14-15 in the LET counts
def expected_let(t, a, box, r_out):
    """N_local, N_soft, N_hard of one domain from whole-array predicates (no walk)"""
    lo, hi = box[:3].astype(F), box[3:].astype(F)
    nlo, nhi = a["nlo"].astype(F), a["nhi"].astype(F)
    inside = np.all(nlo >= lo, axis=1) & np.all(nhi < hi, axis=1)
    touches = np.all(nhi >= lo, axis=1) & np.all(nlo < hi, axis=1)
    r2 = _point_box_d2(a["com_m"][:, :3].astype(F), lo, hi)                 # r_ib^2
    opened = (r2 < a["ropen2"]) | touches                                    # Eq. 14, or part of it is ours
    cut = (F(r_out) + t.get("bmax").astype(F)).astype(F)
    within = r2 < (cut * cut).astype(F)                                      # Eq. 15
    leaf = a["child"] == NOCHILD
    parent = a["parent"].astype(np.int64)
    reach = _reached(parent, opened & ~inside & ~leaf)
    # the hard LET follows the same walk but a node survives only if it and all its ancestors pass Eq. 15
    alive = np.zeros(t.nn, bool)
    alive[0] = within[0]
    for k in range(1, t.nn):
        alive[k] = alive[parent[k]] and within[k]
    n_local = int(a["count"][reach & inside].sum())
    sent = reach & ~inside & ~opened
    n_soft, n_hard = int(sent.sum()), int((sent & alive).sum())
    ps = t.get("pos_sorted")[:, :3].astype(F)
    for k in np.nonzero(reach & ~inside & opened & leaf)[0]:
        seg = ps[a["first"][k]:a["first"][k] + a["count"][k]]
        mine = np.all(seg >= lo, axis=1) & np.all(seg < hi, axis=1)
        d2 = _point_box_d2(seg, lo, hi)
        n_local += int(mine.sum()); n_soft += int((~mine).sum())
        if alive[k]:
            n_hard += int((~mine & (d2 < F(r_out) * F(r_out))).sum())
    return n_local, n_soft, n_hard


def test_let_counts_are_what_eq14_eq15_define():
    cfg = CONFIGS[0].with_(n=6000, mac=1, r_out=0.2, r_in=0.02)
    pos, _ = make_ic(cfg.kind, cfg.n, 41)
    t = O.Tree(pos, O.params_from(cfg))
    a = _arrays(t)
    boxes = virtual_domains(pos, 2, 2, 2, seed=3)
    got = t.let_count(boxes)
    for j in (0, 3, 7):
        assert tuple(int(v) for v in got[j]) == expected_let(t, a, boxes[j], cfg.r_out)


# ---------------------------------------------------------------- the mutants
MUTANTS = {
    "swapped glo/ghi in dist2_box_com": (
        "        float u = t->glo[3 * g + a] - c;\n        float w = c - t->ghi[3 * g + a];",
        "        float u = t->ghi[3 * g + a] - c;\n        float w = c - t->glo[3 * g + a];"),
    "box centre instead of the centre of mass": (
        "        float c = t->com_m[4 * k + a];\n        float u = t->glo[3 * g + a] - c;",
        "        float c = 0.5f * (t->nlo[3 * k + a] + t->nhi[3 * k + a]);\n        float u = t->glo[3 * g + a] - c;"),
}


def _build_mutant(tmp_path, old, new):
    here = os.path.dirname(os.path.abspath(O.__file__))
    src = open(os.path.join(here, "hyb_oracle.c")).read()
    assert src.count(old) == 1, "the oracle source changed: update the mutation"
    (tmp_path / "hyb_oracle.c").write_text(src.replace(old, new))
    (tmp_path / "hyb_oracle.h").write_text(open(os.path.join(here, "hyb_oracle.h")).read())
    lib = str(tmp_path / "libmutant.so")
    subprocess.run(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", lib,
                    str(tmp_path / "hyb_oracle.c"), "-lm"], check=True)
    M = C.CDLL(lib)
    M.orc_tree_build.restype = C.c_void_p
    M.orc_tree_build.argtypes = [C.c_int64, C.c_void_p, C.POINTER(O.OrcParams)]
    M.orc_tree_free.argtypes = [C.c_void_p]
    return M


@pytest.mark.parametrize("name", sorted(MUTANTS))
def test_mutants_are_caught(name, tmp_path):
    """a plausible mistake in rule (a) must fail the set comparison (the real oracle passes it above)"""
    M = _build_mutant(tmp_path, *MUTANTS[name])
    M.orc_walk_lists.restype = C.c_int
    M.orc_walk_lists.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                 C.c_int64, C.c_void_p]
    cfg = CONFIGS[0].with_(hard_cut=0)
    pos, _ = make_ic(cfg.kind, cfg.n, cfg.seed)
    P = O.params_from(cfg)
    t = O.Tree(pos, P)                       # tree arrays do not depend on the walk tests
    a = _arrays(t)
    p4 = np.ascontiguousarray(pos, dtype=np.float32)
    h = M.orc_tree_build(cfg.n, p4.ctypes.data_as(C.c_void_p), C.byref(P))

    def mutant_lists(mode, g):
        cells = np.empty(t.nn, np.uint32); parts = np.empty(t.n, np.uint32); hard = np.empty(t.n, np.uint8)
        nc, npt = C.c_int64(), C.c_int64()
        rc = M.orc_walk_lists(h, mode, g, cells.ctypes.data_as(C.c_void_p), t.nn, C.byref(nc),
                              parts.ctypes.data_as(C.c_void_p), hard.ctypes.data_as(C.c_void_p), t.n, C.byref(npt))
        assert rc == 0
        return cells[:nc.value].copy(), parts[:npt.value].copy(), hard[:npt.value].astype(bool)

    bad = check_tree_lists(mutant_lists, a, t.ng, cfg.r_out, 5)
    M.orc_tree_free(h)
    assert bad > 0, f"mutant '{name}' was not caught"


def test_let_mutant_is_caught(tmp_path):
    """the same for Eq. 14: r_ib measured with the domain faces swapped"""
    M = _build_mutant(tmp_path, "                float u = lo[a] - c, w = c - hi[a];",
                      "                float u = hi[a] - c, w = c - lo[a];")
    M.orc_let_count.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    cfg = CONFIGS[0].with_(n=6000, mac=1, r_out=0.2, r_in=0.02)
    pos, _ = make_ic(cfg.kind, cfg.n, 41)
    P = O.params_from(cfg)
    t = O.Tree(pos, P)
    a = _arrays(t)
    boxes = virtual_domains(pos, 2, 2, 2, seed=3)
    p4 = np.ascontiguousarray(pos, dtype=np.float32)
    h = M.orc_tree_build(cfg.n, p4.ctypes.data_as(C.c_void_p), C.byref(P))
    out = np.zeros((len(boxes), 3), np.uint64)
    M.orc_let_count(h, len(boxes), boxes.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p))
    M.orc_tree_free(h)
    assert any(tuple(int(v) for v in out[j]) != expected_let(t, a, boxes[j], cfg.r_out) for j in (0, 3, 7))
