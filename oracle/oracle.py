"""ctypes wrapper around oracle/libhyb_oracle.so (argument marshalling only).

TEST INFRASTRUCTURE: see oracle/hyb_oracle.h for what each call computes and the PAPER.md
passage it follows.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build

MODE_HYBRID, MODE_HARD, MODE_NORMAL = 0, 1, 2


class OrcParams(C.Structure):
    _fields_ = [("G", C.c_float), ("eps", C.c_float), ("theta", C.c_float), ("a_err", C.c_float),
                ("r_in", C.c_float), ("r_out", C.c_float), ("dt_soft", C.c_float),
                ("n_sub", C.c_int32), ("leaf_max", C.c_int32), ("group_max", C.c_int32),
                ("mac", C.c_int32), ("kfunc", C.c_int32), ("split", C.c_int32), ("grouping", C.c_int32), ("hard_tree", C.c_int32),
                ("hard_cut", C.c_int32)]


def params_from(cfg, **over) -> OrcParams:
    """cfg: any object with the workloads.Config attribute names."""
    d = {f: getattr(cfg, f) for f, _ in OrcParams._fields_}
    d.update(over)
    if d["grouping"] == 2:       # "auto" is a scheduling choice of hyb_step; a tree built on request uses reading 1
        d["grouping"] = 1
    return OrcParams(**d)


_lib = None


def lib():
    global _lib
    if _lib is None:
        import os
        L = C.CDLL(build(sanitize=os.environ.get("HYB_ORACLE_SANITIZE") == "1"))
        L.orc_K.restype = C.c_double
        L.orc_K.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int]
        L.orc_rb.restype = C.c_double
        L.orc_rb.argtypes = [C.c_double] * 3
        L.orc_tree_build.restype = C.c_void_p
        L.orc_tree_build.argtypes = [C.c_int64, C.c_void_p, C.POINTER(OrcParams)]
        L.orc_tree_free.argtypes = [C.c_void_p]
        L.orc_tree_nn.restype = C.c_int64
        L.orc_tree_nn.argtypes = [C.c_void_p]
        L.orc_tree_ng.restype = C.c_int64
        L.orc_tree_ng.argtypes = [C.c_void_p]
        L.orc_tree_get.restype = C.c_int64
        L.orc_tree_get.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int64]
        L.orc_walk_counts.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 3
        L.orc_walk_counts_sel.argtypes = [C.c_void_p, C.c_int, C.c_int64] + [C.c_void_p] * 4
        L.orc_let_count.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        L.orc_walk_lists.restype = C.c_int
        L.orc_walk_lists.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.c_void_p, C.c_int64, C.c_void_p,
                                     C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        L.orc_forces.argtypes = [C.c_void_p, C.c_int, C.c_int64] + [C.c_void_p] * 5
        L.orc_direct.argtypes = [C.c_int64, C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_float, C.c_int,
                                 C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_step.restype = C.c_int
        L.orc_step.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(OrcParams), C.c_int32,
                               C.c_void_p, C.c_void_p, C.c_int]
        L.orc_energy.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_float,
                                 C.c_void_p, C.c_void_p]
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def K(r, r_in, r_out, kfunc=0):
    return lib().orc_K(float(r), float(r_in), float(r_out), int(kfunc))


def rb(bmax, B2, a_err):
    return lib().orc_rb(float(bmax), float(B2), float(a_err))


def num_threads():
    return lib().orc_num_threads()


_GET = {  # name -> (selector, dtype, per-item width, which count)
    "keys": (1, np.uint64, 1, "n"), "perm": (2, np.uint32, 1, "n"), "keys_sorted": (3, np.uint64, 1, "n"),
    "pos_sorted": (4, np.float32, 4, "n"), "level": (5, np.uint8, 1, "nn"), "first": (6, np.uint32, 1, "nn"),
    "count": (7, np.uint32, 1, "nn"), "child": (8, np.uint32, 1, "nn"), "nchild": (9, np.uint8, 1, "nn"),
    "parent": (10, np.uint32, 1, "nn"), "level_offset": (11, np.uint32, 23, "one"),
    "com_m": (12, np.float32, 4, "nn"), "ropen2": (13, np.float32, 1, "nn"), "nlo": (14, np.float32, 3, "nn"),
    "nhi": (15, np.float32, 3, "nn"), "M64": (16, np.float64, 1, "nn"), "C64": (17, np.float64, 3, "nn"),
    "B2": (18, np.float64, 1, "nn"), "bmax": (19, np.float64, 1, "nn"), "gfirst": (20, np.uint32, 1, "ng"),
    "gcount": (21, np.uint32, 1, "ng"), "glo": (22, np.float32, 3, "ng"), "ghi": (23, np.float32, 3, "ng"),
    "bbox": (24, np.float32, 6, "one"), "root_L": (25, np.float64, 1, "one"),
}


class Tree:
    """T2-T11 on pos4 float32 [n,4] in the caller's order."""

    def __init__(self, pos4: np.ndarray, params: OrcParams):
        pos4 = np.ascontiguousarray(pos4, dtype=np.float32)
        assert pos4.ndim == 2 and pos4.shape[1] == 4
        self.n = pos4.shape[0]
        self.params = params
        self._h = lib().orc_tree_build(self.n, _p(pos4), C.byref(params))
        if not self._h:
            raise ValueError("orc_tree_build: invalid input")
        self.nn = lib().orc_tree_nn(self._h)
        self.ng = lib().orc_tree_ng(self._h)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.orc_tree_free(self._h)
            self._h = None

    def get(self, name: str) -> np.ndarray:
        sel, dt, w, which = _GET[name]
        cnt = {"n": self.n, "nn": self.nn, "ng": self.ng, "one": 1}[which]
        out = np.empty((cnt, w) if w > 1 else (cnt,), dtype=dt)
        got = lib().orc_tree_get(self._h, sel, _p(out), out.nbytes)
        assert got == out.nbytes, (name, got, out.nbytes)
        return out[0] if which == "one" and w > 1 else out

    def walk_counts(self, mode: int, gsel=None):
        if gsel is not None:
            gsel = np.ascontiguousarray(gsel, dtype=np.int64)
            k = len(gsel)
            nc = np.zeros(k, np.uint32); npart = np.zeros(k, np.uint32); nh = np.zeros(k, np.uint32)
            lib().orc_walk_counts_sel(self._h, mode, k, _p(gsel), _p(nc), _p(npart), _p(nh))
            return nc, npart, nh
        nc = np.zeros(self.ng, np.uint32); npart = np.zeros(self.ng, np.uint32); nh = np.zeros(self.ng, np.uint32)
        lib().orc_walk_counts(self._h, mode, _p(nc), _p(npart), _p(nh))
        return nc, npart, nh

    def walk_lists(self, mode: int, g: int):
        cc, cp = self.nn, self.n
        cells = np.empty(cc, np.uint32); parts = np.empty(cp, np.uint32); hard = np.empty(cp, np.uint8)
        ncell = C.c_int64(); npart = C.c_int64()
        rc = lib().orc_walk_lists(self._h, mode, g, _p(cells), cc, C.byref(ncell), _p(parts), _p(hard), cp,
                                  C.byref(npart))
        assert rc == 0
        return cells[:ncell.value].copy(), parts[:npart.value].copy(), hard[:npart.value].astype(bool)

    def let_count(self, boxes: np.ndarray) -> np.ndarray:
        """boxes float32 [P,6] (lo xyz, hi xyz) -> uint64 [P,3] = N_local, N_soft, N_hard per domain"""
        boxes = np.ascontiguousarray(boxes, dtype=np.float32)
        out = np.zeros((boxes.shape[0], 3), np.uint64)
        lib().orc_let_count(self._h, boxes.shape[0], _p(boxes), _p(out))
        return out

    def forces(self, mode: int, gsel=None):
        """-> a_soft, a_hard float64 [n,3] in SORTED order, interactions (soft, hard)."""
        a_s = np.zeros((self.n, 3)); a_h = np.zeros((self.n, 3))
        i_s = C.c_double(); i_h = C.c_double()
        if gsel is not None:
            gsel = np.ascontiguousarray(gsel, dtype=np.int64)
            lib().orc_forces(self._h, mode, len(gsel), _p(gsel), _p(a_s), _p(a_h), C.byref(i_s), C.byref(i_h))
        else:
            lib().orc_forces(self._h, mode, 0, None, _p(a_s), _p(a_h), C.byref(i_s), C.byref(i_h))
        return a_s, a_h, (i_s.value, i_h.value)


def direct(pos4, G, eps, r_in=0.0, r_out=0.0, kfunc=0, sel=None):
    """Brute-force Eq. 1-2 (and its K split) -> a_tot, a_hard, a_soft float64 [nsel,3]."""
    pos4 = np.ascontiguousarray(pos4, dtype=np.float32)
    n = pos4.shape[0]
    if sel is None:
        nsel, selp = n, None
    else:
        sel = np.ascontiguousarray(sel, dtype=np.int64); nsel, selp = len(sel), _p(sel)
    at = np.zeros((nsel, 3)); ah = np.zeros((nsel, 3)); as_ = np.zeros((nsel, 3))
    lib().orc_direct(n, _p(pos4), G, eps, r_in, r_out, kfunc, nsel, selp, _p(at), _p(ah), _p(as_))
    return at, ah, as_


def step(x, v, m, params: OrcParams, ncycles=1, a_soft=None, a_hard=None):
    """T16 on fp64 state (in place).  Returns (a_soft, a_hard) valid for the final x."""
    assert x.dtype == np.float64 and v.dtype == np.float64 and x.flags.c_contiguous and v.flags.c_contiguous
    m = np.ascontiguousarray(m, dtype=np.float32)
    n = x.shape[0]
    valid = a_soft is not None and a_hard is not None
    if not valid:
        a_soft = np.zeros((n, 3)); a_hard = np.zeros((n, 3))
    rc = lib().orc_step(n, _p(x), _p(v), _p(m), C.byref(params), ncycles, _p(a_soft), _p(a_hard), int(valid))
    if rc != 0:
        raise ValueError("orc_step failed")
    return a_soft, a_hard


def energy(x, v, m, G, eps):
    x = np.ascontiguousarray(x, dtype=np.float64); v = np.ascontiguousarray(v, dtype=np.float64)
    m = np.ascontiguousarray(m, dtype=np.float32)
    k = C.c_double(); w = C.c_double()
    lib().orc_energy(x.shape[0], _p(x), _p(v), _p(m), G, eps, C.byref(k), C.byref(w))
    return k.value, w.value
