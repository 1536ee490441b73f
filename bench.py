#!/usr/bin/env python
"""bench.py -- two-component D3Q19 MLUPS on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]
                    [--shard replicas|slab]

A "step" is one pass of the whole hot path (SURVEY.md §8a rows a0-a7 except on-demand
diagnostics) over all fluid nodes of the workload.  Default workload: BASELINE.json config 4, the
256^3 sandstone-like mask the north_star quotes its roofline target on.  Inputs are seeded and
synthetic (workloads/generators.py); they stand in for the paper's Bentheimer image.

N > 1 (launched by torch.distributed.run, one rank per GPU): the path shards by z-slabs
(SURVEY.md §8e), so by default ONE box -- config 5, the 512^3 throughput workload, unless --config
says otherwise; the z-open configs 3 and 4 work too -- is cut into N slabs, one per rank, and
stepped by lbm_slab_step with the psi-plane and 5-population halo exchanges as NCCL send/recv on a
side stream ("scaling": "strong").  Rank 0 first times the same box
unsharded on its own GPU (config.single_gpu_ms_per_step_same_workload), so the N = 1 and N > 1
lines are comparable.  --shard replicas runs N independent copies of the single-GPU workload
instead (no data-path collective, "scaling": "weak").  NCCL's INIT log goes to
bench_nccl.<host>.<pid>.log beside the script (NCCL_DEBUG=INFO unless the environment says otherwise).

--impl reference times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the
same workload on the host cores; it is a deliberately slow program, reported as a baseline.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

BYTES_PER_UPDATE_STEP = 472      # 3 x 152 B populations + 8 B psi write + 8 B read
BYTES_PER_UPDATE_COLLIDE = 312   # fused pass alone: 152 read + 8 psi + 152 write
BYTES_PER_UPDATE_DENSITY = 160   # density pass alone: 152 read + 8 write


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=None, choices=[1, 2, 3, 4, 5],
                    help="default: 4 on one GPU (the headline workload), 5 for the sharded run")
    ap.add_argument("--size", type=int, default=None, help="override the box edge (debugging)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="lbm_options field, e.g. --opt graph=0 --opt keep_psi_mb=0 (repeatable)")
    ap.add_argument("--clock-interval-ms", type=float, default=2.0,
                    help="NVML sampling period of clocks and throttle reasons during the timed region")
    ap.add_argument("--no-single", action="store_true",
                    help="sharded run: skip the unsharded reference timing on rank 0")
    ap.add_argument("--shard", default=None, choices=["replicas", "slab"],
                    help="default: slab when WORLD_SIZE > 1, else the plain single-GPU step")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            with open(path) as fh:
                return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def workload(args):
    from workloads import make_config
    c = make_config(args.config, size=args.size)
    if args.config in (1,):
        c["params"]["storage_bits"] = 32  # throughput is quoted on the fp32 production build
    return c


def cpu_sample(cfg, edge=128):
    """Bounded sample of the workload for the CPU oracle: the leading edge^3 corner of the same
    mask and state (end layers re-cleared when z is open so the crop is a valid open box)."""
    m = cfg["mask"]
    e = min(edge, m.shape[0])
    sl = (slice(0, e),) * 3
    mask = np.ascontiguousarray(m[sl]).copy()
    rA = np.ascontiguousarray(cfg["rhoA"][sl]).copy()
    rB = np.ascontiguousarray(cfg["rhoB"][sl]).copy()
    if cfg["params"]["z_open"] and e < m.shape[0]:
        rA[-8:] = np.where(mask[-8:] == 0, rA[-8:], rA[-9].max())
        rB[-8:] = np.where(mask[-8:] == 0, rB[-8:], rB[-9].min())
        mask[-8:] = 0
    return mask, rA, rB, f"leading {e}^3 corner of the {m.shape[0]}^3 mask"


def time_oracle(cfg, steps, warmup, budget_s=15.0):
    from oracle import LbmRef, threads
    mask, rA, rB, what = cpu_sample(cfg)
    p = dict(cfg["params"])
    o = LbmRef(mask, p)
    o.set_density(rA, rB)
    t0 = time.perf_counter()
    o.step(max(1, warmup))
    per = (time.perf_counter() - t0) / max(1, warmup)
    n = steps if steps is not None else max(1, min(200, int(budget_s / max(per, 1e-3))))
    t0 = time.perf_counter()
    o.step(n)
    dt = time.perf_counter() - t0
    mlups = o.num_fluid * n / dt / 1e6
    return dict(value=mlups, unit="MLUPS", cores=threads(), kind="oracle",
                sample=f"{what}: {o.num_fluid} fluid nodes x {n} steps, fp64 dense, OpenMP",
                ms_per_step=1e3 * dt / n, steps=n)


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index, interval=0.002):
        super().__init__(daemon=True)
        self.interval = interval   # a 20-step timed region is 7 ms: sample every 2 ms
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.interval)

    def result(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def aggregate_over_ranks(local_ms, units_per_rank, world, device):
    """Max-over-ranks time and whole-job throughput (units of all ranks / that time)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item())
    return ms, world * units_per_rank / (ms * 1e-3) / 1e6


def source_sha16():
    """First 16 hex digits of the SHA-256 over the CUDA path's sources: identifies the build an
    ncu capture under profiles/ belongs to."""
    import hashlib
    h = hashlib.sha256()
    for f in ("kernels.cuh", "lbm.cu", "geometry.cpp", "geometry.hpp", "torch_shim.cpp"):
        with open(os.path.join(ROOT, "paper_2207_01534_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(workload_name, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload_name` from
    the committed `ncu --set full` capture of THIS build (profiles/ncu_traffic.csv, rows keyed by
    source_sha16), else None: a capture of another build says nothing about this one."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None
    sha = source_sha16()
    with open(path) as fh:
        for line in fh:
            if line.startswith("#"):
                continue
            f = [x.strip() for x in line.split(", ")]     # kernel names hold commas, no ", "
            if len(f) == 4 and f[0] == sha and f[1] == workload_name and f[2] == kernel:
                return float(f[3])
    return None


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores, rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    if args.config is None:   # the arm the driver compares with: same workload as ours for this N
        args.config = 5 if (int(os.environ.get("WORLD_SIZE", "1")) > 1 and args.shard != "replicas") else 4
    cfg = workload(args)
    steps = args.steps if args.steps is not None else None
    warm = args.warmup if args.warmup is not None else 1
    r = time_oracle(cfg, steps, warm)
    line = {"impl": "reference", "metric": "two_component_d3q19_mlups", "value": r["value"],
            "unit": "MLUPS", "n_gpus": args.gpus, "steps": r["steps"], "warmup": warm,
            "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "sample": r["sample"]},
            "cpu_baseline": {"value": r["value"], "unit": "MLUPS", "cores": r["cores"],
                             "kind": "oracle", "sample": r["sample"]},
            "e2e": {"value": r["value"], "unit": "MLUPS", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2207_01534_b200 import Lbm

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    K = args.steps if args.steps is not None else 500
    W = args.warmup if args.warmup is not None else 20
    cfg = workload(args)
    opts = {k: (v if not v.lstrip("-").isdigit() else int(v))
            for k, v in (kv.split("=", 1) for kv in args.opt)}
    sim = Lbm(cfg["mask"], cfg["params"], options=opts or None)
    sim.set_density(cfg["rhoA"], cfg["rhoB"])
    nf = sim.num_fluid
    mem = sim.memory_bytes()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: W warm-up steps, then exactly K steps between events
    sim.step(W)
    barrier()
    sampler = ClockSampler(local, args.clock_interval_ms * 1e-3)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    sim.step(K)
    e1.record()
    barrier()
    sampler.stop_flag = True
    sampler.join()
    ms_total, value = aggregate_over_ranks(e0.elapsed_time(e1), nf * K, world, "cuda")
    _, launches = sim.last_step_profile()
    mass, _ = sim.diagnostics()          # fails loudly on a non-finite state

    # ---- per-kernel durations: a second pass of K steps with CUDA events around every launch
    sim.set_profiling(True)
    sim.step(K)
    kms, _ = sim.last_step_profile()
    sim.set_profiling(False)
    peak, peak_src = measured_peaks()
    t_col = kms["collide_stream"] / K * 1e-3
    achieved = BYTES_PER_UPDATE_COLLIDE * nf / t_col / 1e9
    kname = ("k_collide_stream_bulk<float,128,7,1,1>" if cfg["params"]["storage_bits"] == 32
             else "k_collide_stream_bulk<double,128,2,0,1>")
    roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak,
                "traffic": ncu_traffic(cfg["name"] if args.size is None else None, kname),
                "traffic_source": "profiles/ncu_traffic.csv, build " + source_sha16(),
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": BYTES_PER_UPDATE_COLLIDE * nf,
                "kernel_ms_per_launch": {k: v / K for k, v in kms.items()},
                "step_algorithmic_gbs": BYTES_PER_UPDATE_STEP * nf / (ms_total / K * 1e-3) / 1e9,
                "step_frac_of_peak": BYTES_PER_UPDATE_STEP * nf / (ms_total / K * 1e-3) / 1e9 / peak,
                "step_frac_of_8TBs": BYTES_PER_UPDATE_STEP * nf / (ms_total / K * 1e-3) / 1e9 / 8000.0}

    # ---- end to end through the public API with HOST buffers: upload the initial state, run
    # K steps, download both density fields; copies are inside the timed region.
    e2e = None
    if not args.no_e2e:
        # host buffers are PINNED (page-locked) numpy views of torch tensors, so the copies the
        # C ABI makes from/to them run at PCIe speed
        pin = {k: torch.empty(cfg["mask"].shape, dtype=torch.float64, pin_memory=True).numpy()
               for k in ("inA", "inB", "rhoA", "rhoB")}
        pin["inA"][...] = cfg["rhoA"]
        pin["inB"][...] = cfg["rhoB"]
        out = {"rhoA": pin["rhoA"], "rhoB": pin["rhoB"]}

        def job():
            sim.set_density(pin["inA"], pin["inB"])
            sim.step(K)
            sim.get_macroscopic(fields=("rhoA", "rhoB"), out=out)
            torch.cuda.synchronize()

        # one untimed job first: the staging buffers of set_density / get_macroscopic (0.6 GB from
        # the caching allocator) are then warm, as in any job after the first; cold, the first
        # cudaMalloc alone took up to 70 ms of a 20-step job on some boxes
        job()
        barrier()
        t0 = time.perf_counter()
        job()
        dt = torch.tensor([time.perf_counter() - t0], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(dt, op=dist.ReduceOp.MAX)
        nbytes = 2 * cfg["mask"].size * 8
        e2e = {"value": world * nf * K / float(dt.item()) / 1e6, "unit": "MLUPS",
               "h2d_bytes_per_step": nbytes / K, "d2h_bytes_per_step": nbytes / K,
               "job": f"lbm_set_density (pinned host f64) + lbm_step({K}) + "
                      f"lbm_get_macroscopic(rhoA,rhoB) to pinned host; {nbytes} B each way per job; "
                      "second of two identical jobs (the first warms the allocator)"}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        r = time_oracle(cfg, None, 1)
        cpu = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}

    if rank == 0:
        line = {"metric": "two_component_d3q19_mlups", "value": value, "unit": "MLUPS",
                "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_total / K,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32" if cfg["params"]["storage_bits"] == 32 else "f64",
                "data": "synthetic",
                "config": {"workload": cfg["name"], "box": list(cfg["mask"].shape[::-1]),
                           "fluid_nodes": nf, "wall_solid_nodes": sim.num_wall_solid,
                           "porosity": cfg["porosity"], "parallelism": f"replicas x{world}",
                           "l2": "populations (2 x %.0f MB) exceed the 126 MB L2; no flush needed"
                                 % (mem["populations"] / 2e6),
                           "device_bytes": mem},
                "clocks": sampler.result(), "e2e": e2e, "gpu_launches": launches,
                "roofline": roofline, "cpu_baseline": cpu,
                "mass_check": [float(mass[0]), float(mass[1])]}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_slab(args):
    """--shard slab: one z-periodic box cut into WORLD_SIZE z-slabs (strong scaling)."""
    import torch
    import torch.distributed as dist
    from paper_2207_01534_b200.slab import SlabLbm

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    K = args.steps if args.steps is not None else 200
    W = args.warmup if args.warmup is not None else 20
    cfg = workload(args)
    total_nf = int((cfg["mask"] == 0).sum())

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # the same box, unsharded, on rank 0's GPU: what the sharded number is to be compared with
    single_ms = None
    if rank == 0 and not args.no_single:
        from paper_2207_01534_b200 import Lbm
        ref = Lbm(cfg["mask"], cfg["params"])
        ref.set_density(cfg["rhoA"], cfg["rhoB"])
        ref.step(5)
        torch.cuda.synchronize()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        ref.step(min(K, 50))
        r1.record()
        torch.cuda.synchronize()
        single_ms = r0.elapsed_time(r1) / min(K, 50)
        ref.close()
        torch.cuda.empty_cache()
    barrier()
    sim = SlabLbm(cfg["mask"], cfg["params"], rank=rank, world=world)
    sim.set_density(cfg["rhoA"], cfg["rhoB"])
    one = sim.sims[0]

    sim.step(W)
    barrier()
    one.set_profiling(False)             # restarts the launch counter
    sampler = ClockSampler(local, args.clock_interval_ms * 1e-3)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    sim.step(K)
    e1.record()
    barrier()
    sampler.stop_flag = True
    sampler.join()
    t = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    value = total_nf * K / (ms_total * 1e-3) / 1e6
    _, launches = one.last_step_profile()
    mass, _ = sim.diagnostics()
    one.set_profiling(True)
    sim.step(K)
    kms, _ = one.last_step_profile()
    one.set_profiling(False)
    peak, peak_src = measured_peaks()
    t_col = kms["collide_stream"] / K * 1e-3
    achieved = BYTES_PER_UPDATE_COLLIDE * one.num_owned / t_col / 1e9
    roofline = {"bound": "hbm", "kernel": "k_collide_stream_bulk<float,128,7,1,1>",
                "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": BYTES_PER_UPDATE_COLLIDE * one.num_owned,
                "kernel_ms_per_launch": {("halo_pack_unpack" if k == "open_planes" else k): v / K
                                         for k, v in kms.items()},
                "note": "rank 0's slab"}
    e2e = None
    if not args.no_e2e:
        barrier()
        t0 = time.perf_counter()
        sim.set_density(cfg["rhoA"], cfg["rhoB"])
        sim.step(K)
        out = sim.get_macroscopic(("rhoA", "rhoB"))
        torch.cuda.synchronize()
        dt = torch.tensor([time.perf_counter() - t0], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(dt, op=dist.ReduceOp.MAX)
        z0, z1 = sim.ranges[rank]
        up = 2 * (z1 - z0 + 4) * cfg["mask"][0].size * 8
        down = sum(v.nbytes for v in out.values())
        e2e = {"value": total_nf * K / float(dt.item()) / 1e6, "unit": "MLUPS",
               "h2d_bytes_per_step": up / K, "d2h_bytes_per_step": down / K,
               "job": f"per rank: lbm_set_density of the local box (host f64) + {K} sharded steps + "
                      "lbm_get_macroscopic(rhoA,rhoB) of the owned planes"}
    if rank == 0:
        line = {"metric": "two_component_d3q19_mlups", "value": value, "unit": "MLUPS",
                "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_total / K,
                "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": "f32" if cfg["params"]["storage_bits"] == 32 else "f64",
                "data": "synthetic",
                "config": {"workload": cfg["name"], "box": list(cfg["mask"].shape[::-1]),
                           "fluid_nodes": total_nf, "porosity": cfg["porosity"],
                           "parallelism": f"z-slabs x{world}", "slab_z_ranges": sim.ranges,
                           "slab_step": ("lbm_slab_step (NCCL send/recv inside the library)"
                                         if sim.native else "sequenced from Python (RingTransport)"),
                           "single_gpu_ms_per_step_same_workload": single_ms,
                           "l2": "populations exceed the 126 MB L2 at the default size; no flush"},
                "clocks": sampler.result(), "e2e": e2e, "gpu_launches": launches,
                "roofline": roofline, "cpu_baseline": None,
                "mass_check": [float(mass[0]), float(mass[1])]}
        print(json.dumps(line), flush=True)
    sim.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        world = int(os.environ.get("WORLD_SIZE", "1"))
        shard = a.shard or ("slab" if world > 1 else "replicas")
        if shard == "slab":
            if a.config is None:
                a.config = 5
            if world > 1:
                os.environ.setdefault("NCCL_DEBUG", "INFO")
                os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
                os.environ.setdefault("NCCL_DEBUG_FILE", os.path.join(ROOT, "bench_nccl.%h.%p.log"))
            run_slab(a)
        else:
            if a.config is None:
                a.config = 4
            run_ours(a)
