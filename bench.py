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



def whole_job_value(world: int, units_per_rank: int, ms_per_step_max_over_ranks: float) -> float:
    """metric of the whole job: units all ranks processed / the slowest rank's time (Mrays/s)"""
    return world * units_per_rank / (ms_per_step_max_over_ranks * 1e-3) / 1e6


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """max of a per-rank scalar over all ranks (identity for a single process); works with nccl and gloo"""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


NCU_METRICS = {  # name in the roofline object -> ncu metric (raw page)
    "l1_wavefronts": "l1tex__data_pipe_lsu_wavefronts.sum",
    "l1_sectors_global_ld": "l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum",
    "l2_sectors": "lts__t_sectors_srcunit_tex.sum",          # sectors the L1s requested from L2
    "dram_bytes_read": "dram__bytes_read.sum",
    "dram_bytes_write": "dram__bytes_write.sum",
    "tensor_pipe_pct": "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
    "duration_us_under_ncu": "gpu__time_duration.sum",
}
_UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "sector": 1.0, "": 1.0, "%": 1.0, "us": 1.0,
               "ns": 1e-3, "ms": 1e3, "inst": 1.0, "cycle": 1.0}


def ncu_counts(cfg_id: int, enc: str) -> dict | None:
    """Per-launch counters of the dominant kernel from the committed `ncu --set full` export
    profiles/fused_cfg<id>_r2_raw.csv (made with `bench.py --config <id> --profile-only`, see the .md beside it)."""
    import csv
    f = ROOT / "profiles" / (f"fused_cfg{cfg_id}_r2_raw.csv" if enc == "compose" else f"fused_cfg{cfg_id}_{enc}_r2_raw.csv")
    if not f.exists():
        return None
    rows = list(csv.reader(f.open()))
    hdr, units, vals = rows[0], rows[1], rows[2]
    out = {"file": str(f.relative_to(ROOT))}
    run = f.with_name(f.name.replace("_raw.csv", "_run.txt"))        # the --profile-only line of the captured run
    if run.exists():
        out["hit_rays_per_launch"] = json.loads(run.read_text())["hit_rays_per_launch"]
    for key, metric in NCU_METRICS.items():
        if metric in hdr:
            i = hdr.index(metric)
            out[key] = float(vals[i].replace(",", "")) * _UNIT_SCALE.get(units[i], 1.0)
    # the LSU data-pipe wavefront count is exported per L1 (one per SM) as an average
    per_sm, n_sm = "SM_A.TriageCompute.l1tex__data_pipe_lsu_wavefronts.avg", "device__attribute_multiprocessor_count"
    if "l1_wavefronts" not in out and per_sm in hdr and n_sm in hdr:
        out["l1_wavefronts"] = float(vals[hdr.index(per_sm)].replace(",", "")) * float(vals[hdr.index(n_sm)])
    return out


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


def cpu_baseline(cfg: I.Config, variant: str, budget_s: float = 12.0) -> dict:
    """The oracle as it stands on this box's host cores: one core on a bounded, evenly spread
    sample of the frame, then the same single-threaded function over disjoint ray ranges on every core this
    process may use (oracle/pool.py)."""
    from oracle.pool import OraclePool, cpu_model, n_cores
    run = OracleRun(cfg, variant)
    o, d, stride = run.sample(4096)
    t = run.time_query(o, d)                         # calibration pass
    n_sample = int(min(len(run.origin), max(4096, 4096 * budget_s / max(t, 1e-3))))
    n_sample = 1 << int(np.floor(np.log2(n_sample)))
    o, d, stride = run.sample(n_sample)
    t1 = run.time_query(o, d)
    one = len(o) / t1 / 1e6
    cores = n_cores()
    with OraclePool(cfg.nv, run.occ, run.pose, run.lat, run.params) as pool:
        oa, da, stride_a = run.sample(min(len(run.origin), n_sample * min(cores, 16)))
        pool.query(oa[:4096], da[:4096], occlusion_only=cfg.occlusion_only)      # workers up, libraries loaded
        t0 = time.perf_counter()
        pool.query(oa, da, occlusion_only=cfg.occlusion_only)
        ta = time.perf_counter() - t0
    return {"value": len(oa) / ta / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu_model": cpu_model(),
            "one_core": {"value": one, "unit": UNIT, "cores": 1,
                         "sample": f"every {stride:.1f}th ray of the frame ({len(o)} rays, hits and misses), {t1:.1f} s"},
            "sample": f"every {stride_a:.1f}th ray of the frame ({len(oa)} rays, hits and misses) split over {cores} worker "
                      f"processes, each running the single-threaded oracle/nif_oracle.c as it stands (gcc -O2, fp32), {ta:.1f} s"}


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
    # every rank traces the whole workload (the same seeded frame: independent replicas) = weak scaling
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
    # (no per-kernel events in here: those are collected in a separate pass below)
    sampler = ClockSampler(physical_gpu_index(local_rank))
    launches0 = nif.nif_kernel_launch_count()
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    sync_all()
    sampler.start()
    marks[0].record()
    for i in range(args.steps):
        step()
        marks[i + 1].record()
    sync_all()
    clocks = sampler.stop()
    elapsed_ms = marks[0].elapsed_time(marks[-1])
    step_ms = [marks[i].elapsed_time(marks[i + 1]) for i in range(args.steps)]
    launches = nif.nif_kernel_launch_count() - launches0
    elapsed_ms = max_over_ranks(elapsed_ms, dist if world > 1 else None, dev)
    ms_per_step = elapsed_ms / args.steps
    value = whole_job_value(world, n_total, ms_per_step)
    launches_per_query = 1 if batched else cfg.n_poses     # per-kernel times below are per query launch

    # ---- per-kernel times: the same steps again with the library's event hooks switched on -------
    nif.nif_profile_enable(True)
    for _ in range(max(3, min(args.steps, 10))):
        step()
    prof = nif.nif_profile_read()
    nif.nif_profile_enable(False)
    if args.profile_only:
        if args.with_probe and nif.nif_net_uses_tensor_cores(net):
            for _ in range(4):                         # the MLP-only probe instantiation, for an ncu capture of it
                for p in poses:
                    ws = nif.nif_query(p["bvh"], net, p["o"], p["d"], out, workspace=ws, flags=flags | nif.NIF_PROBE_SKIP_GATHER)
            torch.cuda.synchronize()
        if rank == 0:
            print(json.dumps({"profile_only": True, "config": workload_name(cfg), "ms_per_step": ms_per_step,
                              "hit_rays_per_step": n_hit, "hit_rays_per_launch": n_hit / launches_per_query,
                              "encode_mlp_ms": prof["network_ms"] / max(prof["n_queries"], 1),
                              "traverse_ms": prof["traverse_ms"] / max(prof["n_queries"], 1)}), flush=True)
        if world > 1:
            dist.destroy_process_group()
        return

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
        for _ in range(3):                             # the probe is its own kernel instantiation: warm it up first
            for p in poses:
                ws = nif.nif_query(p["bvh"], net, p["o"], p["d"], out, workspace=ws, flags=flags | nif.NIF_PROBE_SKIP_GATHER)
        torch.cuda.synchronize()
        nif.nif_profile_enable(True)
        for _ in range(10):
            for p in poses:
                ws = nif.nif_query(p["bvh"], net, p["o"], p["d"], out, workspace=ws, flags=flags | nif.NIF_PROBE_SKIP_GATHER)
        pr = nif.nif_profile_read()
        nif.nif_profile_enable(False)
        mlp_probe = pr["network_ms"] / max(pr["n_queries"], 1)          # per nif_query launch = per pose
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
    e2e_s = max_over_ranks(e2e_s, dist if world > 1 else None, dev)
    e2e_value = whole_job_value(world, n_total, e2e_s / e2e_steps * 1e3)
    # the same with the compact return (ids/t for every ray, head rows for hit rays only)
    hit_ray_h = torch.empty(n_per_pose, dtype=torch.int32).pin_memory()
    stage = nif.Stage(max(1, args.chunk // 2))          # less to copy back per chunk: shorter chunks pipeline better
    for p in poses:
        nif.nif_query_host_compact(p["bvh"], net, stage, p["o_h"], p["d_h"], out_h, hit_ray_h, flags=flags)
    sync_all()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        for p in poses:
            nif.nif_query_host_compact(p["bvh"], net, stage, p["o_h"], p["d_h"], out_h, hit_ray_h, flags=flags)
    e2ec_s = max_over_ranks(time.perf_counter() - t0, dist if world > 1 else None, dev)
    e2ec_value = whole_job_value(world, n_total, e2ec_s / e2e_steps * 1e3)
    work = algorithmic_work(cfg)
    h2d = n_total * work["hbm_bytes_per_ray_in"]
    d2h = n_total * work["hbm_bytes_per_ray_out"]

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (fused encode+MLP), measured live -------------------
    # The kernel is a gather machine: its binding units are the L1/LSU data pipe (wavefronts: a gather by 32
    # lanes into 32 different lines costs 32 of them) and the L2 (HBM for config 4) sector path behind it.
    # Ceilings are measured live with the library's two probes; the kernel's own wavefront / sector / DRAM
    # counts per launch come from the committed ncu export under profiles/ (scaled by hit rays per launch).
    peaks = measured_peaks()
    nq = max(prof["n_queries"], 1)
    net_ms = prof["network_ms"] / nq                    # average launch duration, CUDA events
    trav_ms = prof["traverse_ms"] / nq
    hits_per_launch = n_hit / launches_per_query
    table_bytes = params.table_storage().nbytes
    l2_resident = table_bytes <= (64 << 20)              # 126 MB L2: a 32 MiB table stays resident, 512 MiB does not
    smem_kernel = 140 * 1024                             # one block per SM with the fused kernel's carve-out
    pbuf = torch.empty((32 << 20) if l2_resident else (512 << 20), dtype=torch.uint8, device=dev)
    probe_l1 = nif.nif_probe_gather(pbuf[:32 << 20], smem_bytes=smem_kernel, mode=0)    # L1 wavefront ceiling
    # L2 -> SM sector rate: the better of the two request shapes at full occupancy (random single sectors reach
    # ~285 G/s, random whole lines ~245 G/s on this part)
    probe_l2 = max((nif.nif_probe_gather(pbuf[:32 << 20], smem_bytes=0, mode=m) for m in (0, 1)), key=lambda r: r["sectors_per_s"])
    probe_hbm = None if l2_resident else nif.nif_probe_gather(pbuf, smem_bytes=0, mode=1)   # HBM random-sector rate
    del pbuf
    useful_gbs = hits_per_launch * work["useful_gather_bytes"] / (net_ms * 1e-3) / 1e9
    tensor_tfs = hits_per_launch * work["mlp_flops_per_hit_ray"] / (net_ms * 1e-3) / 1e12
    counts = ncu_counts(cfg.cfg_id, args.enc)
    is_tc = (not (flags & nif.NIF_ENGINE_FFMA)) and cfg.net.dtype == "f16" and nif.nif_net_uses_tensor_cores(net)
    roofline = {"kernel": "k_fused_encode_mlp (tcgen05)" if is_tc else "k_encode_mlp_ffma",
                "avg_launch_ms": net_ms, "share_of_step": net_ms * launches_per_query / ms_per_step,
                "algorithmic": f"{work['gathers_per_hit_ray']} gathers x {work['useful_gather_bytes'] // work['gathers_per_hit_ray']} B "
                               f"per hit ray x {hits_per_launch:.0f} hit rays per launch (SURVEY 8(d).2)",
                "useful_gather_gbs": useful_gbs,
                "ceilings": {
                    "l1_wavefronts_per_s": probe_l1["sectors_per_s"],
                    "l1_wavefronts_source": "measured live: nif_probe_gather mode 0 (every lane its own 128 B line of a 32 MiB "
                                            "L2-resident buffer, one block per SM with 140 KB of shared memory like the kernel)",
                    "l2_sectors_per_s": probe_l2["sectors_per_s"],
                    "l2_sectors_source": "measured live: the better of nif_probe_gather mode 0 (random single sectors) and mode 1 (warp-"
                                         "coalesced random 128 B lines) over a 32 MiB L2-resident buffer, 64 warps per SM, no shared memory",
                    "hbm_random_sectors_per_s": probe_hbm["sectors_per_s"] if probe_hbm else None,
                    "hbm_random_sectors_source": "measured live: nif_probe_gather mode 1 over a 512 MiB buffer (HBM-resident like "
                                                 "the table)" if probe_hbm else None,
                    "hbm_copy_gbs": peaks["hbm_gbs"], "hbm_copy_source": f"{peaks['source']} (MEASURED_PEAKS.json)"}}
    if counts and "l1_wavefronts" in counts:
        # per-launch counts of THIS launch = ncu's counts scaled by hit rays (the capture was made on the same workload)
        k = hits_per_launch / counts.get("hit_rays_per_launch", hits_per_launch)
        wf, l2s = counts["l1_wavefronts"] * k, counts.get("l2_sectors", 0.0) * k
        dram = (counts.get("dram_bytes_read", 0.0) + counts.get("dram_bytes_write", 0.0)) * k
        units = {"l1-wavefronts": (wf, probe_l1["sectors_per_s"]), "l2-sectors": (l2s, probe_l2["sectors_per_s"]),
                 "hbm-copy-bytes": (dram / 32.0, peaks["hbm_gbs"] * 1e9 / 32.0)}
        if probe_hbm:
            units["hbm-random-sectors"] = (dram / 32.0, probe_hbm["sectors_per_s"])
        t_unit = {name: c / r for name, (c, r) in units.items()}
        bound = max(t_unit, key=t_unit.get)
        roofline.update({
            "bound": bound, "achieved": units[bound][0] * 32 / (net_ms * 1e-3) / 1e9, "peak": units[bound][1] * 32 / 1e9,
            "unit": "GB/s", "frac": t_unit[bound] / (net_ms * 1e-3), "traffic": dram,
            "frac_by_unit": {name: t / (net_ms * 1e-3) for name, t in t_unit.items()},
            "counts_per_launch": {"l1_wavefronts": wf, "l1_sectors_global_ld": counts.get("l1_sectors_global_ld", 0.0) * k,
                                  "l2_sectors_requested_by_l1": l2s, "dram_bytes": dram, "per_hit_ray": {
                                      "l1_wavefronts": wf / max(hits_per_launch, 1), "l1_sectors": counts.get("l1_sectors_global_ld", 0.0) * k / max(hits_per_launch, 1),
                                      "l2_sectors": l2s / max(hits_per_launch, 1), "dram_bytes": dram / max(hits_per_launch, 1)}},
            "counts_source": counts["file"],
            "what": "for each unit on the gather path: the time it needs for this launch's own count at its measured ceiling, over "
                    "the event-timed launch duration; `bound` is the unit with the largest such fraction and achieved / peak are "
                    "its traffic in GB/s (32 B per wavefront or sector)"})
    else:
        roofline.update({"bound": "l1-wavefronts", "achieved": useful_gbs, "peak": probe_l1["gbps"], "unit": "GB/s",
                         "frac": useful_gbs / probe_l1["gbps"], "traffic": None,
                         "what": "no ncu export for this configuration under profiles/: useful gather bytes over the divergent-"
                                 "gather ceiling (a lower bound of the true fraction: binned rays share sectors)"})
    roofline["tensor"] = {"bound": "tensor", "achieved": tensor_tfs, "peak": peaks["tf_sustained"], "unit": "TFLOP/s",
                          "frac": tensor_tfs / peaks["tf_sustained"], "peak_source": f"{peaks['source']} bf16 sustained (fp16 same pipe)"}
    roofline["hbm_io"] = {"bound": "hbm", "achieved": ((n_total / launches_per_query) * (work["hbm_bytes_per_ray_in"] + work["hbm_bytes_per_ray_out"]))
                          / ((net_ms + trav_ms) * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                          "what": "compulsory ray input / output bytes of the whole query over its duration",
                          "peak_source": f"{peaks['source']} copy bandwidth"}
    roofline["hbm_io"]["frac"] = roofline["hbm_io"]["achieved"] / peaks["hbm_gbs"]
    if mlp_probe:
        hits_probe = n_hit / cfg.n_poses                 # the probe runs one nif_query per pose
        tf = hits_probe * work["mlp_flops_per_hit_ray"] / (mlp_probe * 1e-3) / 1e12
        roofline["tensor_mlp_only_probe"] = {
            "what": "the PROBE instantiation of the same kernel (NIF_PROBE_SKIP_GATHER): constant A operand, no table "
                    "gathers; MLP flops of the real network / event-timed kernel duration, launch and pipeline fill included",
            "avg_launch_ms": mlp_probe, "achieved": tf, "peak": peaks["tf_burst"], "unit": "TFLOP/s", "frac": tf / peaks["tf_burst"],
            "peak_source": f"{peaks['source']} bf16 burst (fp16 same pipe)"}
    kernels = {"traverse_ms": trav_ms, "encode_mlp_ms": net_ms, "traverse_share": trav_ms * launches_per_query / ms_per_step,
               "queries_per_step": launches_per_query,
               "bvh_build_ms_per_pose": float(np.median(build_ms)),
               "bvh_refit_ms_per_pose": float(np.median(refit_ms))}

    base = cpu_baseline(cfg, args.params) if (world == 1 and not args.no_cpu_baseline) else None
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step,
            "ms_per_step_median": float(np.median(step_ms)), "ms_per_step_best": float(np.min(step_ms)),
            "higher_is_better": True,
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
                    "api": "nif_query_host (pinned host buffers, chunked, 3 streams)", "steps": e2e_steps,
                    "compact": {"value": e2ec_value, "unit": UNIT, "h2d_bytes_per_step": h2d,
                                "d2h_bytes_per_step": n_total * 12 + n_hit * (4 + work["hbm_bytes_per_ray_out"] - 12),
                                "api": "nif_query_host_compact: ids and t for every ray, head outputs for hit rays only"}},
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
    ap.add_argument("--profile-only", action="store_true",
                    help="warm-up + a few steps of the query only (no probes, e2e or CPU baseline): the command the "
                         "ncu captures under profiles/ were made with")
    ap.add_argument("--with-probe", action="store_true", help="with --profile-only: also launch the MLP-only probe kernel")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` run plainly: become N ranks (one per GPU) under torch.distributed.run
        import subprocess
        port = 29500 + (os.getpid() % 2000)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), str(Path(__file__).resolve()), *sys.argv[1:]]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
