#!/usr/bin/env python
"""bench.py -- Mrays/s of the neural intersection query (BASELINE.json `metric`) on N B200s.

One "step" = one pass of the whole hot path (traverse -> map back -> encode -> MLP -> decode,
SURVEY.md section 8(a)) over one synthetic frame of BASELINE.json configs[1]: 1920x1080 primary
rays against the 64^3 blob object bent with k = 0.8, network L=16 T=2^19 F=2 B=6, 3x64 fp16 MLP.
Inputs are seeded and synthetic (nif_inputs/).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

N > 1: launched by torch.distributed.run, one rank per GPU.  Rays are independent, so every rank
traces its own full frame (weak scaling, no data-path collective); the
timed region is bracketed by a barrier + synchronize and the maximum over ranks is reported.

The JSON line carries `roofline` (dominant kernel = fused encode+MLP, against the measured
random-sector gather rate; also the tensor-pipe and HBM views), `cpu_baseline` (the oracle on
this box's host cores, bounded sample) and `e2e` (nif_query_host: pinned host buffers, copies in
the timed region).  `--impl reference` times the CPU oracle instead (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import nif_inputs as I  # noqa: E402

METRIC = "Mrays/s neural intersection query on 1 B200; tensor-pipe % of peak (MLP)"
UNIT = "Mrays/s"

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the
# `ncu --set full` capture named beside it (profiles/); None until a capture exists.
NCU_TRAFFIC = {
    # config id: (bytes per launch, profile file)
    1: (33_850_000, "profiles/fused_encode_mlp_r1.md"),
}


def measured_peaks() -> dict:
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return {"hbm_gbs": d["hbm_gbs"], "tf_burst": d["bf16_tflops"], "tf_sustained": d["bf16_tflops_sustained"],
                "source": "measured"}
    return {"hbm_gbs": 6650.0, "tf_burst": 1590.0, "tf_sustained": 1400.0, "source": "fallback"}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.004):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.nv = None

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
                 "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80)}
        get = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
            getattr(nv, "nvmlDeviceGetCurrentClocksThrottleReasons")
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                mask = int(get(self.h))
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def stop(self) -> dict:
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ------------------------------------------------------------------------------------------
# workload description and algorithmic work
# ------------------------------------------------------------------------------------------
def algorithmic_work(cfg: I.Config) -> dict:
    n = cfg.net
    gathers = 2 * (1 if n.enc_mode == "concat" else n.samples) * n.levels * 8
    elem = 2 if n.dtype == "f16" else 4
    dims = n.layer_dims()
    if cfg.occlusion_only:
        dims = dims[:-1] + [(1, n.width)]
    macs = sum(a * b for a, b in dims)
    return {"gathers_per_hit_ray": gathers, "useful_gather_bytes": gathers * n.feat * elem,
            "sector_gather_bytes": gathers * 32, "mlp_flops_per_hit_ray": 2 * macs,
            "hbm_bytes_per_ray_in": 24, "hbm_bytes_per_ray_out": 12 + (4 if cfg.occlusion_only else 48)}


def workload_name(cfg: I.Config) -> str:
    enc = ", concatenation encoding" if cfg.net.enc_mode == "concat" else ""
    return f"configs[{cfg.cfg_id}] {cfg.name}: {cfg.nv}^3 voxels, {cfg.n_poses} pose(s) x {cfg.rays_per_pose} rays{enc}"


def configured(args) -> I.Config:
    cfg = I.get_config(args.config)
    if args.enc == "concat":                       # SURVEY 8(f) f3 variant, not the headline
        from dataclasses import replace
        cfg = replace(cfg, net=replace(cfg.net, enc_mode="concat"))
    return cfg


# ------------------------------------------------------------------------------------------
# the CPU oracle, timed as it stands (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------
class OracleRun:
    def __init__(self, cfg: I.Config, variant: str):
        from oracle import Oracle
        self.cfg = cfg
        self.orc = Oracle()
        self.occ = I.occupancy(cfg)
        self.pose = I.poses(cfg)[0]
        self.params = I.net_params(cfg, variant)
        self.lat = self.orc.deform_lattice(cfg.nv, float(self.pose[0]), float(self.pose[1]))
        self.bvh = self.orc.bvh_build(cfg.nv, self.occ, self.lat)
        lo, hi = self.bvh.bounds()
        self.origin, self.direction = I.rays(cfg, 0, lo, hi)

    def sample(self, n_sample: int):
        n = len(self.origin)
        n_sample = min(n_sample, n)
        idx = (np.arange(n_sample, dtype=np.int64) * n) // n_sample       # evenly spread over the frame
        return np.ascontiguousarray(self.origin[idx]), np.ascontiguousarray(self.direction[idx]), n / n_sample

    def time_query(self, o, d) -> float:
        t0 = time.perf_counter()
        self.orc.query(self.cfg.nv, self.occ, self.lat, self.bvh, self.pose, self.params, o, d,
                       occlusion_only=self.cfg.occlusion_only)
        return time.perf_counter() - t0


def cpu_baseline(cfg: I.Config, variant: str, budget_s: float = 15.0) -> dict:
    run = OracleRun(cfg, variant)
    o, d, stride = run.sample(4096)
    t = run.time_query(o, d)                         # calibration pass
    n_sample = int(min(len(run.origin), max(4096, 4096 * budget_s / max(t, 1e-3))))
    n_sample = 1 << int(np.floor(np.log2(n_sample)))
    o, d, stride = run.sample(n_sample)
    t = run.time_query(o, d)
    return {"value": len(o) / t / 1e6, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"every {stride:.1f}th ray of the frame ({len(o)} rays, hits and misses), "
                      f"single thread, {t:.1f} s; oracle/nif_oracle.c as it stands (gcc -O2, fp32)"}


def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = configured(args)
    run = OracleRun(cfg, args.params)
    o, d, stride = run.sample(args.ref_sample)
    for _ in range(args.warmup):
        run.time_query(o[:1024], d[:1024])
    times = [run.time_query(o, d) for _ in range(args.steps)]
    t = float(np.mean(times))
    value = len(o) / t / 1e6
    sample = (f"each step = every {stride:.1f}th ray of the frame ({len(o)} rays), single thread; "
              "oracle/nif_oracle.c as it stands")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "params": args.params},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------
# our arm: the CUDA path through the C ABI
# ------------------------------------------------------------------------------------------
def run_ours(args) -> None:
    import torch
    import torch.distributed as dist

    import paper_2604_24666_b200 as nif

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback "
                         "(use --impl reference for the CPU oracle)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)

    cfg = configured(args)
    flags = nif.NIF_OCCLUSION_ONLY if cfg.occlusion_only else 0
    if args.engine == "ffma":
        flags |= nif.NIF_ENGINE_FFMA
    occ = I.occupancy(cfg)
    pose_list = I.poses(cfg)
    params = I.net_params(cfg, args.params)
    net = nif.nif_net_create(params.shape, params.level_res, torch.from_numpy(params.table_storage()).to(dev),
                             [torch.from_numpy(w).to(dev) for w in params.weights_storage()])
    occ_d = torch.from_numpy(occ).to(dev)

    # one BVH + one ray batch per pose ("for each deformation pose, we build a simple BVH");
    # every rank traces the whole workload with its own ray seed offset = weak scaling
    poses, build_ms = [], []
    for pi in range(cfg.n_poses):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        bvh = nif.nif_build_deformed_bvh(cfg.nv, occ_d, float(pose_list[pi][0]), float(pose_list[pi][1]),
                                         max_occupied=int(occ.sum()))
        e1.record(); torch.cuda.synchronize()
        build_ms.append(e0.elapsed_time(e1))
        info = bvh.info()
        o, d = I.rays(cfg, pi, info["lo"], info["hi"])
        poses.append({"bvh": bvh, "o_h": torch.from_numpy(o).pin_memory(), "d_h": torch.from_numpy(d).pin_memory(),
                      "o": torch.from_numpy(o).to(dev), "d": torch.from_numpy(d).to(dev)})
    # refit (same voxel set, new pose): back to the first pose's neighbour and home again, timed
    refit_ms = []
    for pi in range(cfg.n_poses):
        th, kk = float(pose_list[pi][0]), float(pose_list[pi][1])
        poses[pi]["bvh"].refit(th * 0.5, kk * 0.5)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        poses[pi]["bvh"].refit(th, kk)
        e1.record(); torch.cuda.synchronize()
        refit_ms.append(e0.elapsed_time(e1))
    n_per_pose = cfg.rays_per_pose
    n_total = n_per_pose * cfg.n_poses
    batched = cfg.n_poses > 1 and args.poses == "batched" and not args.walk
    if batched:                                        # one nif_query_poses over the rays of all poses (B:9)
        all_o = torch.cat([p["o"] for p in poses]); all_d = torch.cat([p["d"] for p in poses])
        all_pid = torch.cat([torch.full((n_per_pose,), i, dtype=torch.int32, device=dev) for i in range(cfg.n_poses)])
        all_bvh = [p["bvh"] for p in poses]
        out_all = nif.alloc_outputs(n_total, device=dev)
        ws_all = None
    out = nif.alloc_outputs(n_per_pose, device=dev)
    walk_out = nif.alloc_walk_outputs(n_per_pose, device=dev) if args.walk else None
    ws = None
    ws_multi = None

    def step():
        nonlocal ws, ws_multi, ws_all
        if batched:
            ws_all = nif.nif_query_poses(all_bvh, net, all_o, all_d, all_pid, out_all, workspace=ws_all, flags=flags)
            return
        for p in poses:
            if args.walk:                              # multi-voxel walk, --walk K rounds
                ws_multi = nif.nif_query_multi(p["bvh"], net, p["o"], p["d"], out, walk_out, args.walk,
                                               workspace=ws_multi, flags=flags)
            else:
                ws = nif.nif_query(p["bvh"], net, p["o"], p["d"], out, workspace=ws, flags=flags)

    def sync_all():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    n_hit = 0
    for p in poses:                                    # hit count per pose (workload property)
        w_ = nif.nif_query(p["bvh"], net, p["o"], p["d"], out, workspace=ws, flags=flags)
        n_hit += nif.nif_query_last_hit_count(w_)

    # ---- timed region: K steps, device-timed, inputs resident in HBM -------------------------
    sampler = ClockSampler(physical_gpu_index(local_rank))
    nif.nif_profile_enable(True)
    launches0 = nif.nif_kernel_launch_count()
    sync_all()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    sync_all()
    clocks = sampler.stop()
    elapsed_ms = e0.elapsed_time(e1)
    launches = nif.nif_kernel_launch_count() - launches0
    prof = nif.nif_profile_read()
    nif.nif_profile_enable(False)
    if world > 1:
        t = torch.tensor([elapsed_ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        elapsed_ms = float(t.item())
    ms_per_step = elapsed_ms / args.steps
    value = world * n_total / (ms_per_step * 1e-3) / 1e6
    launches_per_query = 1 if batched else cfg.n_poses     # per-kernel times below are per query launch

    walk_stats = None
    if args.walk:
        torch.cuda.synchronize()
        st = walk_out["status"]; sp = walk_out["steps"]
        walk_stats = {"max_steps": args.walk, "last_pose_status_counts": [int((st == k).sum()) for k in range(3)],
                      "last_pose_network_evals": int(sp.sum()), "last_pose_mean_steps_of_entering_rays":
                      float(sp[sp > 0].float().mean()) if bool((sp > 0).any()) else 0.0}

    # ---- MLP-only probe: same kernel, gathers replaced by a constant A operand (outside the timed region)
    mlp_probe = None
    if rank == 0 and not args.walk and nif.nif_net_uses_tensor_cores(net) and not (flags & nif.NIF_ENGINE_FFMA):
        nif.nif_profile_enable(True)
        for _ in range(5):
            for p in poses:
                ws = nif.nif_query(p["bvh"], net, p["o"], p["d"], out, workspace=ws, flags=flags | nif.NIF_PROBE_SKIP_GATHER)
        pr = nif.nif_profile_read()
        nif.nif_profile_enable(False)
        mlp_probe = pr["network_ms"] / max(pr["n_queries"], 1)
        for p in poses:                                # leave real results in `out`
            ws = nif.nif_query(p["bvh"], net, p["o"], p["d"], out, workspace=ws, flags=flags)
        torch.cuda.synchronize()

    # ---- e2e: same metric through nif_query_host (pinned host buffers, copies timed) ---------
    stage = nif.Stage(args.chunk)
    out_h = nif.alloc_outputs(n_per_pose, pinned_host=True)
    for _ in range(2):
        for p in poses:
            nif.nif_query_host(p["bvh"], net, stage, p["o_h"], p["d_h"], out_h, flags=flags)
    sync_all()
    e2e_steps = max(3, min(args.steps, 10))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        for p in poses:
            nif.nif_query_host(p["bvh"], net, stage, p["o_h"], p["d_h"], out_h, flags=flags)   # synchronises
    e2e_s = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([e2e_s], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e_value = world * n_total * e2e_steps / e2e_s / 1e6
    work = algorithmic_work(cfg)
    h2d = n_total * work["hbm_bytes_per_ray_in"]
    d2h = n_total * work["hbm_bytes_per_ray_out"]

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (fused encode+MLP), measured live -------------------
    peaks = measured_peaks()
    nq = max(prof["n_queries"], 1)
    net_ms = prof["network_ms"] / nq                    # average launch duration, CUDA events
    trav_ms = prof["traverse_ms"] / nq
    hits_per_launch = n_hit / launches_per_query
    table_bytes = params.table_storage().nbytes
    l2_resident = table_bytes <= (64 << 20)              # 126 MB L2: a 32 MiB table stays resident, 512 MiB does not
    probe_bytes = (32 << 20) if l2_resident else (256 << 20)
    probe = nif.nif_probe_gather(torch.from_numpy(params.table_storage()).to(dev).view(torch.uint8).reshape(-1)
                                 if args.probe_table else torch.empty(probe_bytes, dtype=torch.uint8, device=dev))
    useful_gbs = hits_per_launch * work["useful_gather_bytes"] / (net_ms * 1e-3) / 1e9
    gather_gbs = hits_per_launch * work["sector_gather_bytes"] / (net_ms * 1e-3) / 1e9
    tensor_tfs = hits_per_launch * work["mlp_flops_per_hit_ray"] / (net_ms * 1e-3) / 1e12
    traffic = NCU_TRAFFIC.get(cfg.cfg_id, (None, None))
    roofline = {"kernel": "k_fused_encode_mlp (tcgen05)" if not (flags & nif.NIF_ENGINE_FFMA) and cfg.net.dtype == "f16"
                and nif.nif_net_uses_tensor_cores(net) else "k_encode_mlp_ffma",
                "bound": "l2-gather" if l2_resident else "hbm-gather",
                "achieved": useful_gbs, "peak": probe["gbps"], "unit": "GB/s",
                "frac": useful_gbs / probe["gbps"], "traffic": traffic[0],
                "peak_source": f"measured live: nif_probe_gather, independent random 32 B sectors over a "
                               f"{probe_bytes >> 20} MiB buffer ({'L2' if l2_resident else 'HBM'}-resident like the table), all SMs; "
                               "MEASURED_PEAKS.json has no gather figure (its HBM and tensor peaks are in .hbm / .tensor)",
                "algorithmic": f"useful gather bytes (SURVEY 8(d).2): {work['gathers_per_hit_ray']} gathers x "
                               f"{work['useful_gather_bytes'] // work['gathers_per_hit_ray']} B per hit ray x "
                               f"{hits_per_launch:.0f} hit rays per launch",
                "frac_note": "useful bytes delivered per second over the best rate at which the memory system delivers "
                             "32 B sectors; the sectors ncu counted at L2 (profiles/) are within 8 % of the useful bytes "
                             "on config 1 because binned rays share sectors",
                "sector_worst_case": {"achieved": gather_gbs, "frac": gather_gbs / probe["gbps"],
                                      "what": "every lane's gather counted as its own 32 B sector (SURVEY 8(d).2 worst case); "
                                              "exceeds 1 when the 32 rays of a warp share sectors"},
                "avg_launch_ms": net_ms, "share_of_step": net_ms * launches_per_query / ms_per_step,
                "tensor": {"bound": "tensor", "achieved": tensor_tfs, "peak": peaks["tf_sustained"],
                           "unit": "TFLOP/s", "frac": tensor_tfs / peaks["tf_sustained"],
                           "peak_source": f"{peaks['source']} bf16 sustained (fp16 same pipe)"},
                "hbm": {"bound": "hbm", "achieved": ((n_total / launches_per_query) * (work["hbm_bytes_per_ray_in"] + work["hbm_bytes_per_ray_out"]))
                        / ((net_ms + trav_ms) * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                        "peak_source": f"{peaks['source']} copy bandwidth"}}
    roofline["hbm"]["frac"] = roofline["hbm"]["achieved"] / peaks["hbm_gbs"]
    if mlp_probe:
        tf = hits_per_launch * work["mlp_flops_per_hit_ray"] / (mlp_probe * 1e-3) / 1e12
        roofline["tensor_mlp_only_probe"] = {
            "what": "same kernel with NIF_PROBE_SKIP_GATHER: constant A operand, no table gathers; MLP flops of "
                    "the real network / event-timed kernel duration", "avg_launch_ms": mlp_probe,
            "achieved": tf, "peak": peaks["tf_burst"], "unit": "TFLOP/s", "frac": tf / peaks["tf_burst"],
            "peak_source": f"{peaks['source']} bf16 burst (fp16 same pipe)"}
    kernels = {"traverse_ms": trav_ms, "encode_mlp_ms": net_ms, "traverse_share": trav_ms * launches_per_query / ms_per_step,
               "queries_per_step": launches_per_query,
               "bvh_build_ms_per_pose": float(np.median(build_ms)),
               "bvh_refit_ms_per_pose": float(np.median(refit_ms))}

    base = cpu_baseline(cfg, args.params) if (world == 1 and not args.no_cpu_baseline) else None
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f16" if cfg.net.dtype == "f16" else "f32",
            "data": "synthetic",
            "config": {"workload": workload_name(cfg), "params": args.params, "rays_per_step_per_gpu": n_total,
                       "hit_rays_per_step_per_gpu": n_hit, "hit_fraction": n_hit / n_total,
                       "l2": f"no flush: per-step working set (rays 24 B + outputs 60 B per ray + {params.table_storage().nbytes >> 20} MiB table) "
                             "exceeds the 126 MB L2" + ("; the hash table is meant to stay L2-resident between frames"
                                                         if params.table_storage().nbytes <= (64 << 20) else ""),
                       "poses": ("one nif_query_poses over all poses" if batched else "one nif_query per pose"),
                       "parallelism": f"dp{world} (independent frames per rank, no collective)"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "api": "nif_query_host (pinned host buffers, chunked, 3 streams)", "steps": e2e_steps},
            "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline, "kernels": kernels,
            "mhit_rays_per_s": world * n_hit / (ms_per_step * 1e-3) / 1e6}
    if walk_stats is not None:
        line["config"]["walk"] = walk_stats
        line["config"]["workload"] += f", multi-voxel walk max_steps={args.walk}"
    if base is not None:
        line["cpu_baseline"] = base
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (default 1: the headline)")
    ap.add_argument("--params", default="uniform0.1", choices=["uniform0.1", "varpres"])
    ap.add_argument("--engine", default="auto", choices=["auto", "ffma"])
    ap.add_argument("--chunk", type=int, default=1 << 20, help="rays per staging chunk of nif_query_host")
    ap.add_argument("--ref-sample", type=int, default=32768, help="rays per step of --impl reference")
    ap.add_argument("--probe-table", action="store_true", help="run the gather probe over the real table")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--enc", default="compose", choices=["compose", "concat"],
                    help="hybrid-encoding reading: the paper's composition (default, headline) or concatenation")
    ap.add_argument("--poses", default="batched", choices=["batched", "loop"],
                    help="multi-pose configs: one nif_query_poses per step (default) or one nif_query per pose")
    ap.add_argument("--walk", type=int, default=0, help="time nif_query_multi with this max_steps instead of nif_query "
                                                        "(SURVEY 8(f) f1; not the headline; use --params varpres)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
