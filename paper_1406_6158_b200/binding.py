"""ctypes binding of include/hyb.h.  No arithmetic of the method lives here."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIBPATH = os.path.join(HERE, "libhyb.so")

ERR_NAMES = {0: "HYB_OK", -1: "HYB_ERR_INVALID_ARG", -2: "HYB_ERR_WORKSPACE_TOO_SMALL",
             -3: "HYB_ERR_NONFINITE_INPUT", -4: "HYB_ERR_CAPACITY_OVERFLOW", -5: "HYB_ERR_NO_TREE",
             -6: "HYB_ERR_CUDA", -7: "HYB_ERR_INTERNAL"}

# name -> (selector, dtype, items per unit, unit)   unit in {"n", "nn", "ng", "fixed"}
EXPORTS = {
    "counts": (0, np.int64, 8, "fixed"), "keys_sorted": (1, np.uint64, 1, "n"), "perm": (2, np.uint32, 1, "n"),
    "level": (3, np.uint8, 1, "nn"), "first": (4, np.uint32, 1, "nn"), "count": (5, np.uint32, 1, "nn"),
    "child": (6, np.uint32, 1, "nn"), "nchild": (7, np.uint8, 1, "nn"), "parent": (8, np.uint32, 1, "nn"),
    "level_offset": (9, np.uint32, 23, "fixed"), "com_m": (10, np.float32, 4, "nn"),
    "ropen2": (11, np.float32, 1, "nn"), "nlo": (12, np.float32, 4, "nn"), "nhi": (13, np.float32, 4, "nn"),
    "gfirst": (14, np.uint32, 1, "ng"), "gcount": (15, np.uint32, 1, "ng"), "glo": (16, np.float32, 4, "ng"),
    "ghi": (17, np.float32, 4, "ng"), "ncell": (18, np.uint32, 1, "ng"), "npart": (19, np.uint32, 1, "ng"),
    "nhard": (20, np.uint32, 1, "ng"), "interactions": (21, np.uint64, 4, "fixed"),
    "timings": (22, np.float32, 8, "fixed"), "bbox": (23, np.float32, 6, "fixed"), "keys": (24, np.uint64, 1, "n"),
    "M64": (25, np.float64, 1, "nn"), "C64": (26, np.float64, 3, "nn"), "B2": (27, np.float64, 1, "nn"),
    "bmax": (28, np.float64, 1, "nn"),
}


class HybError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERR_NAMES.get(code, code)}: {msg}")
        self.code = code


class HybParams(C.Structure):
    _fields_ = [("G", C.c_float), ("eps", C.c_float), ("theta", C.c_float), ("a_err", C.c_float),
                ("r_in", C.c_float), ("r_out", C.c_float), ("dt_soft", C.c_float),
                ("n_sub", C.c_int32), ("leaf_max", C.c_int32), ("group_max", C.c_int32),
                ("mac", C.c_int32), ("kfunc", C.c_int32), ("split", C.c_int32), ("grouping", C.c_int32), ("hard_tree", C.c_int32), ("hard_refit", C.c_int32),
                ("hard_cut", C.c_int32)]

    @classmethod
    def from_config(cls, cfg, **over):
        d = {f: getattr(cfg, f) for f, _ in cls._fields_}
        d.update(over)
        return cls(**d)


_lib = None


def lib():
    """Load libhyb.so.  Fails loudly if it has not been built: there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIBPATH):
            raise RuntimeError(f"{LIBPATH} is missing: run `python -m paper_1406_6158_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIBPATH)
        vp = C.c_void_p
        L.hyb_workspace_bytes.restype = C.c_size_t
        L.hyb_workspace_bytes.argtypes = [C.c_int64, C.POINTER(HybParams)]
        L.hyb_init.restype = C.c_int
        L.hyb_init.argtypes = [C.POINTER(vp), C.POINTER(HybParams), C.c_int64, vp, vp, vp, vp, vp, vp, C.c_size_t,
                               C.c_int, vp]
        for name in ("hyb_build_tree", "hyb_build_tree_hard", "hyb_refit_tree", "hyb_soft_force", "hyb_hard_force", "hyb_sync"):
            getattr(L, name).restype = C.c_int
            getattr(L, name).argtypes = [vp]
        L.hyb_set_params.restype = C.c_int
        L.hyb_set_params.argtypes = [vp, C.POINTER(HybParams)]
        L.hyb_set_sink_range.restype = C.c_int
        L.hyb_set_sink_range.argtypes = [vp, C.c_int64, C.c_int64]
        L.hyb_kick_drift.restype = C.c_int
        L.hyb_kick_drift.argtypes = [vp, C.c_float, C.c_float, C.c_float]
        L.hyb_step.restype = C.c_int
        L.hyb_step.argtypes = [vp, C.c_int32]
        L.hyb_export.restype = C.c_int
        L.hyb_export.argtypes = [vp, C.c_int32, vp, C.c_size_t, C.POINTER(C.c_size_t)]
        L.hyb_run_host.restype = C.c_int
        L.hyb_run_host.argtypes = [C.POINTER(HybParams), C.c_int64, vp, vp, vp, vp, vp, C.c_int32, C.c_int32, C.c_int, vp]
        L.hyb_energy.restype = C.c_int
        L.hyb_energy.argtypes = [vp, vp]
        L.hyb_let_count.restype = C.c_int
        L.hyb_let_count.argtypes = [vp, C.c_int32, vp, vp]
        L.hyb_energy_noalloc.restype = C.c_int
        L.hyb_energy_noalloc.argtypes = [vp, vp, C.c_int64, C.c_float, C.c_float, C.c_int, vp, vp]
        L.hyb_probe_fp32.restype = C.c_int
        L.hyb_probe_fp32.argtypes = [C.c_int, vp, vp, C.c_size_t, vp]
        L.hyb_run_host_release.restype = None
        L.hyb_run_host_release.argtypes = []
        L.hyb_last_error.restype = C.c_char_p
        L.hyb_last_error.argtypes = [vp]
        L.hyb_free.restype = None
        L.hyb_free.argtypes = [vp]
        _lib = L
    return _lib


def hyb_workspace_bytes(n: int, params: HybParams) -> int:
    return lib().hyb_workspace_bytes(n, C.byref(params))


def hyb_run_host(params: HybParams, pos_m: np.ndarray, vel: np.ndarray, ids: np.ndarray, n_soft_steps: int,
                 device: int = 0, a_soft: np.ndarray | None = None, a_hard: np.ndarray | None = None,
                 acc_valid: bool = False):
    """End-to-end call on HOST (NumPy / pinned torch) buffers; updates pos_m, vel, ids in place and
    returns (a_soft, a_hard, interactions).  acc_valid: a_soft / a_hard hold the accelerations of pos_m (from the
    previous call) and are uploaded instead of being evaluated again.  a_soft / a_hard: optional float32 [n,4] result buffers (pass
    pinned ones to keep the download off the pageable-memory path); allocated here when omitted."""
    n = pos_m.shape[0]
    if a_soft is None:
        a_soft = np.empty((n, 4), np.float32)
    if a_hard is None:
        a_hard = np.empty((n, 4), np.float32)
    for a in (a_soft, a_hard):
        assert a.dtype == np.float32 and a.shape == (n, 4) and a.flags.c_contiguous
    inter = np.zeros(4, np.uint64)
    p = lambda a: C.c_void_p(a.ctypes.data)  # noqa: E731
    rc = lib().hyb_run_host(C.byref(params), n, p(pos_m), p(vel), p(a_soft), p(a_hard), p(ids), n_soft_steps,
                            int(acc_valid), device, p(inter))
    if rc != 0:
        raise HybError(rc, lib().hyb_last_error(None).decode())
    return a_soft, a_hard, inter


def hyb_probe_fp32(device: int = 0):
    """(packed, scalar) FP32 fused multiply-add rate of the device in TFLOP/s (diagnostic; see include/hyb.h)"""
    import torch
    scratch = torch.empty(1 << 20, dtype=torch.float32, device=f"cuda:{device}")
    out = np.zeros(2, np.float64)
    rc = lib().hyb_probe_fp32(device, torch.cuda.current_stream(device).cuda_stream, scratch.data_ptr(), scratch.numel(),
                              C.c_void_p(out.ctypes.data))
    if rc != 0:
        raise HybError(rc, "hyb_probe_fp32")
    return float(out[0]), float(out[1])


def hyb_energy_noalloc(pos_m, vel, G: float, eps: float, out):
    """T, W of the particles in the CUDA tensors pos_m / vel (float32 [n, 4]) into the CUDA tensor out (float64 [2]),
    on torch's current stream, with no allocation and no synchronisation (include/hyb.h); returns out"""
    import torch
    assert pos_m.is_cuda and vel.is_cuda and out.is_cuda and pos_m.is_contiguous() and vel.is_contiguous()
    assert pos_m.dtype == torch.float32 and vel.dtype == torch.float32 and out.dtype == torch.float64 and out.numel() == 2
    assert pos_m.shape == vel.shape and pos_m.shape[1] == 4
    dev = pos_m.device.index
    rc = lib().hyb_energy_noalloc(pos_m.data_ptr(), vel.data_ptr(), pos_m.shape[0], float(G), float(eps), dev,
                                  torch.cuda.current_stream(dev).cuda_stream, out.data_ptr())
    if rc != 0:
        raise HybError(rc, lib().hyb_last_error(None).decode())
    return out


def hyb_run_host_release() -> None:
    lib().hyb_run_host_release()


class Hyb:
    """One hyb context over torch CUDA tensors (float32 [n,4] pos_m / vel, int32 [n] ids)."""

    def __init__(self, params: HybParams, pos_m, vel, ids=None, stream=None):
        import torch
        assert pos_m.is_cuda and pos_m.dtype == torch.float32 and pos_m.shape[1] == 4 and pos_m.is_contiguous()
        assert vel.is_cuda and vel.dtype == torch.float32 and vel.shape == pos_m.shape and vel.is_contiguous()
        self.torch = torch
        self.params = params
        self.n = pos_m.shape[0]
        self.device = pos_m.device
        self.pos_m, self.vel = pos_m, vel
        self.ids = ids if ids is not None else torch.arange(self.n, dtype=torch.int32, device=self.device)
        assert self.ids.dtype == torch.int32 and self.ids.is_contiguous()
        self.a_soft = torch.zeros_like(pos_m)
        self.a_hard = torch.zeros_like(pos_m)
        nbytes = hyb_workspace_bytes(self.n, params)
        if nbytes == 0:
            raise HybError(-1, "invalid parameters")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = C.c_void_p()
        dev_index = self.device.index if self.device.index is not None else torch.cuda.current_device()
        rc = lib().hyb_init(C.byref(self._h), C.byref(params), self.n, pos_m.data_ptr(), vel.data_ptr(),
                            self.a_soft.data_ptr(), self.a_hard.data_ptr(), self.ids.data_ptr(),
                            self.workspace.data_ptr(), nbytes, dev_index, self.stream.cuda_stream)
        if rc != 0:
            raise HybError(rc, lib().hyb_last_error(None).decode())

    def _check(self, rc):
        if rc != 0:
            raise HybError(rc, lib().hyb_last_error(self._h).decode())

    def set_params(self, params: HybParams):
        self._check(lib().hyb_set_params(self._h, C.byref(params)))
        self.params = params

    def build_tree(self):
        self._check(lib().hyb_build_tree(self._h))

    def build_tree_hard(self):
        self._check(lib().hyb_build_tree_hard(self._h))

    def refit_tree(self):
        self._check(lib().hyb_refit_tree(self._h))

    def soft_force(self):
        self._check(lib().hyb_soft_force(self._h))

    def hard_force(self):
        self._check(lib().hyb_hard_force(self._h))

    def set_sink_range(self, first: int, last: int):
        self._check(lib().hyb_set_sink_range(self._h, first, last))

    def kick_drift(self, c_soft: float, c_hard: float, dt: float):
        self._check(lib().hyb_kick_drift(self._h, c_soft, c_hard, dt))

    def step(self, n_soft_steps: int = 1):
        self._check(lib().hyb_step(self._h, n_soft_steps))

    def let_count(self, boxes: np.ndarray) -> np.ndarray:
        """boxes float32 [P,6] (lo xyz, hi xyz) -> uint64 [P,3] = N_local, N_soft, N_hard per virtual domain"""
        boxes = np.ascontiguousarray(boxes, dtype=np.float32)
        out = np.zeros((boxes.shape[0], 3), np.uint64)
        self._check(lib().hyb_let_count(self._h, boxes.shape[0], C.c_void_p(boxes.ctypes.data), C.c_void_p(out.ctypes.data)))
        return out

    def energy(self):
        """(T, W): kinetic and unsplit softened potential energy of the current state, fp64, summed on the device"""
        out = np.zeros(2, np.float64)
        self._check(lib().hyb_energy(self._h, C.c_void_p(out.ctypes.data)))
        return float(out[0]), float(out[1])

    def sync(self):
        self._check(lib().hyb_sync(self._h))

    def export(self, name: str) -> np.ndarray:
        sel, dt, width, unit = EXPORTS[name]
        if unit == "fixed":
            cnt = 1
        else:
            c = self.export("counts")
            cnt = int({"n": c[0], "nn": c[1], "ng": c[2]}[unit])
        out = np.empty((cnt, width) if width > 1 else (cnt,), dtype=dt)
        written = C.c_size_t()
        self._check(lib().hyb_export(self._h, sel, C.c_void_p(out.ctypes.data), out.nbytes, C.byref(written)))
        assert written.value == out.nbytes, (name, written.value, out.nbytes)
        return out[0] if unit == "fixed" else out

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().hyb_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
