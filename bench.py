#!/usr/bin/env python
"""bench.py -- one JSON line for the hybrid tree force path.

A "step" is one soft cycle Delta t_s of the whole hot path on BASELINE.json's N = 2^20 workload
(configs[2]: Hernquist sphere): n tree builds, one fused soft+hard walk, n-1 hard walks, kick/drift.
metric = pairwise interactions evaluated per second (sum over groups of members x list length).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config I]

N > 1 runs under torchrun, one independent replica per rank (the path does not shard: "replicas
only"); value is the whole-job aggregate over ranks, time the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# flop conventions: monopole pair 23 (north_star), K-weighted pairs from the
# instruction list of walk.cu: fused soft+hard pair 43, hard-only pair 36.
FLOP_MONO, FLOP_KFUSED, FLOP_KHARD = 23.0, 43.0, 36.0
N_SM, FP32_LANES = 148, 128          # B200: guide's unit counts


def clock_sampler(stop, out, index):
    """sample SM clock and throttle reasons with NVML while the timed region runs"""
    try:
        import pynvml as nv
        nv.nvmlInit()
        h = nv.nvmlDeviceGetHandleByIndex(index)
        out["sm_max_mhz"] = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        out["ready"].set()
        while not stop.is_set():
            if not out["go"].is_set():
                time.sleep(0.001)
                continue
            out["samples"].append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
            r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
            for bit, nm in names.items():
                if r & bit:
                    out["reasons"].add(nm)
            time.sleep(0.002)
    except Exception as e:  # noqa: BLE001
        out["error"] = repr(e)
        out["ready"].set()


def oracle_sample(cfg, pos, seconds):
    """times the oracle (as it stands) on a bounded sample of the workload: full tree build, then
    the fused soft+hard force evaluation on evenly spaced sink groups for about `seconds`."""
    import numpy as np
    from oracle import oracle as O
    P = O.params_from(cfg)
    t0 = time.perf_counter()
    tree = O.Tree(pos, P)
    t_build = time.perf_counter() - t0
    probe = np.linspace(0, tree.ng - 1, num=min(tree.ng, 256)).astype(np.int64)
    t0 = time.perf_counter()
    _, _, inter = tree.forces(O.MODE_HYBRID, probe)
    t_probe = time.perf_counter() - t0
    want = int(min(tree.ng, max(256, len(probe) * seconds / max(t_probe, 1e-6))))
    gsel = np.unique(np.linspace(0, tree.ng - 1, num=want).astype(np.int64))
    reps = 0
    n_inter = 0.0
    t0 = time.perf_counter()
    while True:
        _, _, inter = tree.forces(O.MODE_HYBRID, gsel)
        n_inter += inter[0]                # pair evaluations: a near pair is on both lists but evaluated once
        reps += 1
        dt = time.perf_counter() - t0
        if dt >= 0.8 * seconds or reps >= 64:
            break
    return {"value": n_inter / dt, "unit": "interactions/s", "cores": O.num_threads(), "kind": "oracle",
            "sample": f"{reps} x fp64 soft+hard force evaluation on {len(gsel)} of {tree.ng} sink groups "
                      f"({n_inter:.3e} interactions in {dt:.2f} s; full tree build {t_build:.2f} s not included)"}, \
        (tree, gsel, n_inter, dt)


def oracle_cycle_split(cfg, pos, vel):
    """one soft cycle of the oracle (as it stands), stage by stage on the full workload: a full tree build and the fused
    soft+hard force evaluation once, a hard-step tree build and a hard-only evaluation once (scaled by n_sub - 1), and the
    kick/drift arithmetic; seconds on the host cores (SURVEY.md 8(d) 'oracle timing')."""
    import numpy as np
    from oracle import oracle as O
    t = {}
    t0 = time.perf_counter(); tree = O.Tree(pos, O.params_from(cfg)); t["build_soft_step_s"] = time.perf_counter() - t0
    t0 = time.perf_counter(); tree.forces(O.MODE_HYBRID); t["soft_step_forces_s"] = time.perf_counter() - t0
    del tree
    gm = max(cfg.group_max // 2, cfg.leaf_max) if cfg.grouping == 2 else cfg.group_max
    t0 = time.perf_counter(); tree = O.Tree(pos, O.params_from(cfg, group_max=gm)); t["build_hard_step_s"] = time.perf_counter() - t0
    t0 = time.perf_counter(); tree.forces(O.MODE_HARD); t["hard_step_forces_s"] = time.perf_counter() - t0
    del tree
    x = pos[:, :3].astype(np.float64); v = vel[:, :3].astype(np.float64); a = np.zeros_like(x)
    t0 = time.perf_counter()
    for _ in range(cfg.n_sub):
        v += 0.5 * a; x += 0.1 * v; v += 0.5 * a
    t["integrate_s"] = time.perf_counter() - t0
    k = cfg.n_sub - 1 if cfg.split else 0
    t["cycle_s"] = (t["build_soft_step_s"] + t["soft_step_forces_s"] + k * (t["build_hard_step_s"] + t["hard_step_forces_s"])
                    + t["integrate_s"])
    t["what"] = (f"1 soft-step (build + fused forces) + {k} hard-steps (build + hard forces), each stage timed once on all "
                 f"{cfg.n} particles; PAPER.md:87, 200")
    return t


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--no-normal", action="store_true", help="skip the normal-tree comparison leg")
    ap.add_argument("--paper-n", type=int, default=None,
                    help="instead of --config: the paper's own recipe (PAPER.md:172-174) for a Plummer model of N particles")
    ap.add_argument("--hard-refit", type=int, default=None, choices=[0, 1],
                    help="1: hard-only substeps refit the boxes instead of rebuilding the tree (not the paper's procedure)")
    ap.add_argument("--hard-tree", type=int, default=None, choices=[0, 1],
                    help="1: the paper's MAC-approximated hard walk instead of the direct hard sum (DESIGN.md R20)")
    ap.add_argument("--hard-cut", type=int, default=None, choices=[0, 1],
                    help="hard list: 0 every particle of the leaves within r_out of the group box, 1 only the particles within r_out of it (DESIGN.md R30)")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: ONE problem with its sinks divided over the ranks (sharded.py, strong scaling) instead of "
                         "independent replicas; unmeasured on hardware, not the headline")
    ap.add_argument("--mac", type=int, default=None, choices=[0, 1],
                    help="opening criterion: 0 theta (the configurations), 1 the paper's absolute MAC with a_err = 2^-8 (Eq. 5-6)")
    ap.add_argument("--grouping", type=int, default=None, choices=[0, 1, 2],
                    help="sink groups: 0 single tree nodes, 1 runs of sibling cells, 2 auto (the configs' default)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    from workloads import CONFIGS, make_ic
    cfg = CONFIGS[args.config]
    if args.paper_n is not None:
        from workloads import paper_params
        cfg = paper_params(args.paper_n, seed=7)
    if args.grouping is not None:
        cfg = cfg.with_(grouping=args.grouping)
    if args.hard_tree is not None:
        cfg = cfg.with_(hard_tree=args.hard_tree)
    if args.hard_refit is not None:
        cfg = cfg.with_(hard_refit=args.hard_refit)
    if args.hard_cut is not None:
        cfg = cfg.with_(hard_cut=args.hard_cut)
    if args.mac is not None:
        cfg = cfg.with_(mac=args.mac)
    config = {"workload": f"{cfg.name}: {cfg.kind} N={cfg.n}, eps={cfg.eps}, theta={cfg.theta}, leaf<={cfg.leaf_max}, "
                          f"group<={cfg.group_max}, r_in={cfg.r_in}, r_out={cfg.r_out}, dt_soft=1/{round(1 / cfg.dt_soft)}, "
                          f"n_sub={cfg.n_sub}, mac={cfg.mac}, grouping={cfg.grouping}, hard_tree={cfg.hard_tree}, hard_refit={cfg.hard_refit}, "
                          f"hard_cut={cfg.hard_cut}, seed {cfg.seed}",
              "step": "one soft cycle: n_sub tree builds + 1 fused soft/hard walk + (n_sub-1) hard walks + kick/drift",
              "l2": "256 MiB L2 flush between timed steps", "replicas": world}

    if args.impl == "reference":
        # the oracle, as it stands, on the host cores; rank 0 only
        if rank != 0:
            return
        pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
        per_step = max(1.0, min(args.cpu_seconds, 120.0 / max(1, args.steps + args.warmup)))
        cb, (tree, gsel, _, _) = oracle_sample(cfg, pos, per_step)
        from oracle import oracle as O
        times, inters = [], []
        for i in range(args.warmup + args.steps):
            t0 = time.perf_counter()
            _, _, inter = tree.forces(O.MODE_HYBRID, gsel)
            dt = time.perf_counter() - t0
            if i >= args.warmup:
                times.append(dt); inters.append(inter[0])
        value = sum(inters) / sum(times)
        cb["value"] = value
        print(json.dumps({"impl": "reference", "metric": "interactions/s", "value": value, "unit": "interactions/s",
                          "n_gpus": 0, "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": 1e3 * sum(times) / len(times), "higher_is_better": True, "scaling": "weak",
                          "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config,
                          "cpu_baseline": cb,
                          "e2e": {"value": value, "unit": "interactions/s", "h2d_bytes_per_step": 0,
                                  "d2h_bytes_per_step": 0}, "gpu_launches": 0}))
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1406_6158_b200 import Hyb, HybParams, hyb_run_host, hyb_probe_fp32

    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl")
    from paper_1406_6158_b200.replicas import replica_seed
    if args.sharded:
        # ---- sink-sharded variant: every rank holds all particles, evaluates its share of the sink
        #      groups, one all-reduce of the accelerations after each force evaluation
        from types import SimpleNamespace
        from paper_1406_6158_b200.sharded import ShardedHyb
        pos, vel = make_ic(cfg.kind, cfg.n, cfg.seed)
        h = Hyb(HybParams.from_config(cfg), torch.from_numpy(pos).cuda(), torch.from_numpy(vel).cuda())
        ar = (lambda t: dist.all_reduce(t)) if world > 1 else (lambda t: None)
        sh = ShardedHyb(h, SimpleNamespace(split=cfg.split, n_sub=cfg.n_sub, dt_soft=cfg.dt_soft), rank, world, ar)
        for _ in range(args.warmup + 1):
            sh.step(1)
        h.sync(); h.export("interactions")
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            sh.step(1)
        e1.record(); h.sync(); torch.cuda.synchronize()
        it = h.export("interactions").astype(np.float64)
        from paper_1406_6158_b200.replicas import aggregate
        ms, _, value = aggregate(e0.elapsed_time(e1), float(it[0] + it[1] - it[2]), device="cuda")
        if rank == 0:
            config["parallelism"] = f"sink-sharded x{world}: replicated particles and tree, all-reduce of a_soft / a_hard"
            print(json.dumps({"metric": "interactions/s", "value": value, "unit": "interactions/s", "n_gpus": world,
                              "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
                              "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
                              "data": "synthetic", "config": config, "note": "variant, unmeasured on more than one GPU"}))
        h.close()
        if world > 1:
            dist.destroy_process_group()
        return
    pos, vel = make_ic(cfg.kind, cfg.n, replica_seed(cfg.seed, rank))      # independent replica per rank
    P = HybParams.from_config(cfg)
    dpos = torch.from_numpy(pos).cuda(); dvel = torch.from_numpy(vel).cuda()
    h = Hyb(P, dpos, dvel)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    h.step(0)                                                   # initial tree + forces (not a timed step)
    for _ in range(args.warmup):
        h.step(1)
    h.export("interactions"); h.export("timings")
    launches0 = int(h.export("counts")[6])

    clk = {"samples": [], "reasons": set(), "ready": threading.Event(), "go": threading.Event()}
    stop = threading.Event()
    th = threading.Thread(target=clock_sampler, args=(stop, clk, local_rank), daemon=True)
    th.start()
    clk["ready"].wait(30.0)                                     # NVML initialised before the timed region starts
    clk["go"].set()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        flush.zero_()                                           # L2 flush, outside the event pair
        a.record()
        h.step(1)
        b.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    stop.set(); th.join()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    inter = h.export("interactions").astype(np.float64)
    stage = h.export("timings").astype(np.float64)
    launches = int(h.export("counts")[6]) - launches0
    from paper_1406_6158_b200.replicas import aggregate
    # pair EVALUATIONS: a near pair of a fused soft+hard walk is on the soft list and on the hard list (inter[0] and
    # inter[1] both count it, inter[2] says how many) but is evaluated once
    total_ms, _, value = aggregate(total_ms, float(inter[0] + inter[1] - inter[2]), device="cuda")     # max over ranks, sum of work

    # ---- roofline of the dominant kernel (the fused soft+hard group walk), rank 0's numbers
    K = args.steps
    soft_ms = stage[1] / K                                       # one launch per step
    fused_hard = inter[2]                                       # hard pairs evaluated inside the soft-step walks
    mono = inter[0] - fused_hard                                # plain monopole pairs (cells + far particles)
    flops = (FLOP_MONO * mono + FLOP_KFUSED * fused_hard) / K
    sm = sorted(clk["samples"])
    sm_mhz = sm[len(sm) // 2] if sm else None
    sm_max = clk.get("sm_max_mhz", 1965)
    peak = N_SM * FP32_LANES * 2 * sm_max * 1e6 / 1e12
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")      # "kernel,dram_bytes_per_launch" from the ncu --set full capture
    if os.path.exists(tpath):
        for line in open(tpath):
            k, _, v = line.strip().partition(",")
            if k == "walk_kernel<HYBRID>":
                traffic = float(v)
    achieved = flops / (soft_ms * 1e-3) / 1e12
    probe = hyb_probe_fp32(local_rank) if rank == 0 else (None, None)      # measured FP32 fused multiply-add rate (not timed)
    roofline = {"bound": "alu", "kernel": "walk_kernel<HYBRID> (fused soft+hard group walk)", "achieved": achieved,
                "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic,
                "peak_source": f"derived: {N_SM} SMs x {FP32_LANES} FP32 lanes x 2 flop x {sm_max} MHz max SM clock "
                               "(MEASURED_PEAKS.json has no FP32 CUDA-core figure)",
                "peak_probe": {"ffma2_tflops": probe[0], "ffma_tflops": probe[1], "frac_of_probe": achieved / probe[0] if probe[0] else None,
                               "what": "hyb_probe_fp32: chains of packed / scalar fused multiply-adds only, measured in this run"},
                "frac_at_sampled_clock": (achieved / (N_SM * FP32_LANES * 2 * sm_mhz * 1e6 / 1e12)) if sm_mhz else None,
                "interactions_per_s": (mono + fused_hard) / K / (soft_ms * 1e-3),
                "flop_per_pair": {"monopole": FLOP_MONO, "k_fused": FLOP_KFUSED, "k_hard": FLOP_KHARD},
                # the hard-only walks: pairs on the hard lists as evaluated (hard_cut = 1: particles within r_out of the group
                # box) and as the leaf-level reading of T13 would list them (every particle of a leaf within r_out)
                "hard_walk": {"interactions_per_s": (inter[1] - fused_hard) / max(stage[2] * 1e-3, 1e-12),
                              "tflops": FLOP_KHARD * (inter[1] - fused_hard) / max(stage[2] * 1e-3, 1e-12) / 1e12,
                              "frac": FLOP_KHARD * (inter[1] - fused_hard) / max(stage[2] * 1e-3, 1e-12) / 1e12 / peak,
                              "frac_leaf_list_count": FLOP_KHARD * inter[3] / max(stage[2] * 1e-3, 1e-12) / 1e12 / peak,
                              "pairs_per_walk": {"evaluated": (inter[1] - fused_hard) / K / max(cfg.n_sub - 1, 1),
                                                 "leaf_list": inter[3] / K / max(cfg.n_sub - 1, 1)}}}
    stages = {"build_ms": stage[0] / K, "soft_ms": soft_ms, "hard_ms": stage[2] / K, "integrate_ms": stage[3] / K}
    # ---- HBM-bound stages: algorithmic bytes over the measured time, against the measured copy peak
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm_peak, hbm_src = 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"
    if os.path.exists(peaks_path):
        hbm_peak, hbm_src = float(json.load(open(peaks_path))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    nodes_per_particle = 0.4
    build_bytes = {"bbox": 16, "keys": 16 + 12, "radix_sort": 8 * (12 + 12), "permute": 4 + 36 + 36,
                   "octree": 16 + nodes_per_particle * 24, "upsweep": 16 + nodes_per_particle * (64 + 56), "groups": 8}
    bpp_build = sum(build_bytes.values())
    bpp_integrate = (96 + (cfg.n_sub - 1) * 80 + 64) if cfg.split else cfg.n_sub * (64 + 64)
    gbs_build = bpp_build * cfg.n * cfg.n_sub / (stages["build_ms"] * 1e-3) / 1e9
    gbs_int = bpp_integrate * cfg.n / (stages["integrate_ms"] * 1e-3) / 1e9
    hbm_stages = {"peak_gbs": hbm_peak, "peak_source": hbm_src,
                  "build": {"bytes_per_particle": bpp_build, "by_stage": build_bytes, "achieved_gbs": gbs_build,
                            "frac": gbs_build / hbm_peak, "radix_sort_share_of_bytes": build_bytes["radix_sort"] / bpp_build},
                  "integrate": {"bytes_per_particle_per_cycle": bpp_integrate, "achieved_gbs": gbs_int, "frac": gbs_int / hbm_peak},
                  "note": "N = 2^20 fits the 126 MB L2 and these stages are latency-bound (about 30 dependent kernels per "
                          "build), so the achieved figure is far below the copy peak; see profiles/r02_profile.md"}

    # ---- end to end through the C-ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if rank == 0 and not args.no_e2e:
        hp = torch.from_numpy(pos).pin_memory(); hv = torch.from_numpy(vel).pin_memory()
        hid = torch.arange(cfg.n, dtype=torch.int32).pin_memory()
        has = torch.empty(cfg.n, 4).pin_memory(); hah = torch.empty(cfg.n, 4).pin_memory()      # results
        e_int, e_t = 0.0, 0.0
        # the state lives in (pinned) host memory between the calls; every timed call is one soft cycle:
        # upload pos / vel / id and the accelerations of the previous call, hyb_step(1), download all five
        hyb_run_host(P, hp.numpy(), hv.numpy(), hid.numpy(), 0, local_rank, has.numpy(), hah.numpy())     # initial forces
        for i in range(2 + 3):
            t0 = time.perf_counter()
            _, _, it = hyb_run_host(P, hp.numpy(), hv.numpy(), hid.numpy(), 1, local_rank, has.numpy(), hah.numpy(),
                                    acc_valid=True)
            dt = time.perf_counter() - t0
            if i >= 2:
                e_int += float(it[0]) + float(it[1]) - float(it[2]); e_t += dt
        n = cfg.n
        e2e = {"value": e_int / e_t, "unit": "interactions/s", "h2d_bytes_per_step": 68 * n,
               "d2h_bytes_per_step": 68 * n, "ms_per_step": 1e3 * e_t / 3,
               "what": "hyb_run_host(acc_valid = 1), one soft cycle per call with the state in pinned host memory: upload "
                       "pos/vel/id/a_soft/a_hard, hyb_step(1), download the same five arrays; wall clock around the call "
                       "(2 untimed calls first; the device buffer is kept between calls)"}

    # ---- the same cycle with a plain (unsplit, theta-only) tree at dt_h: n_sub
    #      builds + n_sub full walks per cycle; reported beside the hybrid to show its compute ratio
    #      (the paper's R_hybrid of about 0.8 is a multi-process wall-clock ratio on other hardware)
    normal = None
    if rank == 0 and not args.no_normal:
        hn = Hyb(HybParams.from_config(cfg, split=0), torch.from_numpy(pos).cuda(), torch.from_numpy(vel).cuda())
        hn.step(0)
        for _ in range(2):
            hn.step(1)
        hn.export("interactions"); hn.export("timings")
        kn = max(2, min(K, 4))
        evn = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(kn)]
        for a, b in evn:
            flush.zero_()
            a.record(); hn.step(1); b.record()
        torch.cuda.synchronize()
        n_ms = sum(a.elapsed_time(b) for a, b in evn) / kn
        n_inter = hn.export("interactions").astype(np.float64)
        n_stage = hn.export("timings").astype(np.float64)
        walk_ms = n_stage[1] / kn / cfg.n_sub                    # one unsplit walk
        normal = {"ms_per_step": n_ms, "interactions_per_s": float(n_inter[0] + n_inter[1]) / kn / (n_ms * 1e-3),
                  "stages": {"build_ms": n_stage[0] / kn, "walk_ms": n_stage[1] / kn, "integrate_ms": n_stage[3] / kn},
                  "walk_kernel": {"ms": walk_ms, "interactions_per_s": n_inter[0] / kn / cfg.n_sub / (walk_ms * 1e-3),
                                  "tflops": FLOP_MONO * n_inter[0] / kn / cfg.n_sub / (walk_ms * 1e-3) / 1e12,
                                  "frac_of_fp32_peak": FLOP_MONO * n_inter[0] / kn / cfg.n_sub / (walk_ms * 1e-3) / 1e12 / peak},
                  "t_hybrid_over_t_normal": (total_ms / K) / n_ms,
                  "hard_walk_over_normal_walk": (stage[2] / K / max(cfg.n_sub - 1, 1)) / walk_ms,
                  "paper_context": "PAPER.md:182 hard kernel ~40 % of a normal-tree force kernel; PAPER.md:216 total time "
                                   "80-90 % of a normal tree (HA-PACS: Tesla M2090 + E5-2670, multi-process)"}
        hn.close()

    # ---- variant, not the headline: hard-only substeps refit the tight boxes instead of rebuilding the tree
    #      (R21: the paper rebuilds; the hard force is the same direct sum either way)
    refit = None
    if rank == 0 and not args.no_normal and cfg.split and not cfg.hard_tree and not cfg.hard_refit and cfg.n_sub > 1:
        hr = Hyb(HybParams.from_config(cfg, hard_refit=1), torch.from_numpy(pos).cuda(), torch.from_numpy(vel).cuda())
        hr.step(0)
        for _ in range(2):
            hr.step(1)
        hr.export("interactions"); hr.export("timings")
        kr = max(2, min(K, 4))
        evr = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(kr)]
        for a, b in evr:
            flush.zero_()
            a.record(); hr.step(1); b.record()
        torch.cuda.synchronize()
        r_ms = sum(a.elapsed_time(b) for a, b in evr) / kr
        r_stage = hr.export("timings").astype(np.float64)
        refit = {"ms_per_step": r_ms, "stages": {"build_or_refit_ms": r_stage[0] / kr, "soft_ms": r_stage[1] / kr,
                                                 "hard_ms": r_stage[2] / kr, "integrate_ms": r_stage[3] / kr},
                 "ratio_to_rebuild": r_ms / (total_ms / K),
                 "what": "hard_refit = 1: one tree build per soft step, n_sub - 1 box refits; same forces up to fp32 summation order"}
        hr.close()

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_baseline, _ = oracle_sample(cfg, pos, args.cpu_seconds)
        if cfg.n <= (1 << 20):
            cpu_baseline["cycle_split"] = oracle_cycle_split(cfg, pos, vel)

    if rank == 0:
        print(json.dumps({
            "metric": "interactions/s", "value": value, "unit": "interactions/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak",
            "stages": stages, "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config,
            "interactions_per_step": {"evaluated": (inter[0] + inter[1] - inter[2]) / K, "soft_lists": inter[0] / K,
                                      "hard_lists": inter[1] / K, "on_both_lists_of_a_fused_walk": inter[2] / K},
            "value_counts": "pair evaluations (a near pair of the fused walk is on both lists and counted once)",
            "roofline": roofline, "hbm_stages": hbm_stages, "normal_tree": normal, "hard_refit_variant": refit, "cpu_baseline": cpu_baseline, "e2e": e2e,
            "gpu_launches": launches,
            "clocks": {"sm_mhz": sm_mhz, "sm_max_mhz": sm_max, "reasons": sorted(clk["reasons"]),
                       "samples": len(sm), **({"error": clk["error"]} if "error" in clk else {})}}))
    h.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
