"""-m gpu, collected last: hyb_energy_noalloc (include/hyb.h) -- the energy diagnostic with its partial sums in a
static device array instead of a context's workspace, for callers that cannot allocate -- against the existing
hyb_energy on the same particles: two calls in a row (the array keeps the first call's contents), the size limit,
and that no device memory is taken."""
import numpy as np
import pytest
import torch

from workloads import CONFIGS, make_ic

pytestmark = pytest.mark.gpu

from gpu_util import make_hyb  # noqa: E402

W_REL = 2e-6          # tests/test_gpu_energy.py: fp32 pair terms against the fp64 sum
T_REL = 1e-12


def _reference(cfg, pos, vel):
    h = make_hyb(cfg, pos, vel)
    t, w = h.energy()
    h.close()
    return t, w


def test_two_calls_in_a_row_match_hyb_energy():
    from paper_1406_6158_b200 import hyb_energy_noalloc
    cfg_a = CONFIGS[0].with_(n=20011, eps=0.01, G=1.0)
    cfg_b = CONFIGS[0].with_(n=777, eps=0.02, G=1.5)          # fewer blocks than the call before: stale partial sums stay behind
    runs = []
    for cfg, kind, seed in ((cfg_a, "hernquist", 5), (cfg_b, "cold_sphere", 6)):
        pos, vel = make_ic(kind, cfg.n, seed)
        runs.append((cfg, pos, vel, _reference(cfg, pos, vel)))
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    for _ in range(2):                                        # a, b, a, b: each call after one of another shape
        for cfg, pos, vel, (t_ref, w_ref) in runs:
            dpos, dvel = torch.from_numpy(pos).cuda(), torch.from_numpy(vel).cuda()
            keep = dpos.clone(), dvel.clone()
            out.fill_(float("nan"))
            hyb_energy_noalloc(dpos, dvel, cfg.G, cfg.eps, out)
            hyb_energy_noalloc(dpos, dvel, cfg.G, cfg.eps, out)      # second call in a row, same stream
            t, w = out.cpu().numpy()
            assert t == pytest.approx(t_ref, rel=T_REL) and w == pytest.approx(w_ref, rel=W_REL)
            assert (t, w) == (t_ref, w_ref)                   # same kernels, same summation order: the same bits
            assert torch.equal(dpos, keep[0]) and torch.equal(dvel, keep[1])      # inputs untouched


def test_no_device_memory_is_taken_and_the_limit_is_reported():
    from paper_1406_6158_b200 import HybError, hyb_energy_noalloc
    from paper_1406_6158_b200.binding import lib
    n = 50000
    pos, vel = make_ic("plummer", n, 3)
    dpos, dvel = torch.from_numpy(pos).cuda(), torch.from_numpy(vel).cuda()
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    hyb_energy_noalloc(dpos, dvel, 1.0, 0.01, out)            # warm: module load, address of the static array
    torch.cuda.synchronize()
    first = out.clone()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        hyb_energy_noalloc(dpos, dvel, 1.0, 0.01, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    assert torch.equal(out, first)
    # beyond the stated maximum: refused before anything is launched, with a message that names the limit
    rc = lib().hyb_energy_noalloc(dpos.data_ptr(), dvel.data_ptr(), 4194304 + 1, 1.0, 0.01, 0,
                                  torch.cuda.current_stream().cuda_stream, out.data_ptr())
    assert rc == -1 and b"HYB_ENERGY_NOALLOC_MAX_N" in lib().hyb_last_error(None)
    with pytest.raises(HybError):
        hyb_energy_noalloc(dpos[:0], dvel[:0], 1.0, 0.01, out)      # n = 0
    torch.cuda.synchronize()
    assert torch.equal(out, first)


def test_largest_size():
    """n = HYB_ENERGY_NOALLOC_MAX_N fits the static array on this device (8192 + 592 + 2 partial sums of 16384)"""
    from paper_1406_6158_b200 import hyb_energy_noalloc
    n = 4194304
    g = torch.Generator(device="cuda").manual_seed(1)
    dpos = torch.rand((n, 4), dtype=torch.float32, device="cuda", generator=g)
    dpos[:, 3] = 1.0 / n
    dvel = torch.zeros_like(dpos); dvel[:, 0] = 1.0
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    hyb_energy_noalloc(dpos, dvel, 1.0, 0.05, out)
    t, w = out.cpu().numpy()
    assert t == pytest.approx(0.5, rel=1e-6)                  # sum 1/2 m v^2 with sum m = 1 (masses rounded to fp32)
    assert -3.0 < w < -0.5                                    # uniform unit cube, unit mass: W = -0.94 G M^2 / L without softening
