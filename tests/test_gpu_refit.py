"""-m gpu: hard_refit / hyb_refit_tree.  A refitted tree (same store order and topology, tight boxes of the
drifted positions) must give the hard force its plain definition: the direct K-weighted sum over every
particle within r_out (Eq. 8), here by brute force in fp64."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from workloads import CONFIGS, make_ic

pytestmark = pytest.mark.gpu

from gpu_util import acc_errors, make_hyb, MAX_TOL, RMS_TOL  # noqa: E402
from test_gpu_configs import _snapshot_parity  # noqa: E402


@pytest.mark.parametrize("n,kind,disp,grouping", [(20011, "plummer", 2e-3, 2), (9973, "hernquist", 5e-3, 0),
                                                   (30000, "cold_sphere", 1e-3, 1)])
def test_refit_hard_force_is_the_direct_sum(n, kind, disp, grouping):
    cfg = CONFIGS[1].with_(n=n, kind=kind, grouping=grouping)
    pos, vel = make_ic(kind, n, 61)
    h = make_hyb(cfg, pos, vel)
    h.build_tree(); h.soft_force(); h.sync()
    # move every particle a little (several substeps' worth of drift), in the store's order
    g = torch.Generator(device="cuda"); g.manual_seed(5)
    h.pos_m[:, :3] += disp * torch.randn((n, 3), generator=g, device="cuda")
    h.refit_tree(); h.hard_force(); h.sync()
    store = h.pos_m.cpu().numpy()
    at, ah, _ = O.direct(store, cfg.G, cfg.eps, cfg.r_in, cfg.r_out)
    rms, mx = acc_errors(h.a_hard.cpu().numpy()[:, :3], ah, at)
    print(rms, mx)
    assert rms < RMS_TOL and mx < MAX_TOL
    # the refitted tree serves the hard force only
    from paper_1406_6158_b200 import HybError
    with pytest.raises(HybError) as ei:
        h.soft_force()
    assert ei.value.code == -5
    h.build_tree(); h.soft_force(); h.sync()             # and a rebuild makes everything valid again
    h.close()


def test_step_with_refit_tracks_step_with_rebuild():
    cfg = CONFIGS[1].with_(n=30011)
    pos, vel = make_ic(cfg.kind, cfg.n, 62)
    out = {}
    for refit in (0, 1):
        h = make_hyb(cfg, pos, vel, hard_refit=refit)
        h.step(3); h.sync()
        ids = h.ids.cpu().numpy().astype(np.int64)
        x = np.empty((cfg.n, 3)); v = np.empty((cfg.n, 3))
        x[ids] = h.pos_m.cpu().numpy()[:, :3]; v[ids] = h.vel.cpu().numpy()[:, :3]
        out[refit] = (x, v)
        if refit:
            print(_snapshot_parity(h, cfg.with_(hard_refit=1)))      # the final tree is a full build again
        h.close()
    # the same forces up to the order of fp32 additions: trajectories agree to rounding level after 3 cycles
    assert np.abs(out[0][0] - out[1][0]).max() < 5e-6 and np.abs(out[0][1] - out[1][1]).max() < 5e-5


def test_refit_errors():
    from paper_1406_6158_b200 import HybError
    cfg = CONFIGS[0].with_(n=800)
    pos, vel = make_ic(cfg.kind, cfg.n, 2)
    h = make_hyb(cfg, pos, vel)
    with pytest.raises(HybError) as ei:
        h.refit_tree()
    assert ei.value.code == -5
    h.close()
    h = make_hyb(cfg, pos, vel, hard_tree=1)
    h.build_tree()
    with pytest.raises(HybError) as ei:
        h.refit_tree()
    assert ei.value.code == -1
    h.close()
    with pytest.raises(HybError):
        make_hyb(cfg, pos, vel, hard_refit=1, hard_tree=1)
