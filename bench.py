"""bench.py — throughput of the geodesic-tracing hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

One "step" = one pass of the whole hot path (work fetch,
pixel map, initial condition, metric + RHS, Runge-Kutta steps with control, termination and
landing, monitors, record store) over one image of the workload, i.e. ONE launch of the
persistent trace kernel through the C-ABI call gp_trace.  The default workload is `headline`:
BASELINE.json configs[1] (Kerr a = 0.9, adaptive Dormand-Prince 5(4), rtol 1e-10) at
1024 x 1024, the configuration BASELINE.json's `metric` is quoted on.

Printed JSON line (rank 0): geodesics/s over all ranks (`value`), the same through
gp_trace_host with pinned host buffers (`e2e`), the ALU roofline of the trace kernel
(`roofline`), the oracle timed on the host cores on a bounded sample (`cpu_baseline`),
the SM clocks sampled during the timed region (`clocks`).

--impl reference times the CPU oracle as it stands (rank 0 only) on the same metric/config.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gp_workloads as W  # noqa: E402

# ---- algorithmic FP64 flop models (+,-,x = 1, FMA = 2, 1/x, sqrt, sin, cos,
# exp, pow = 1 each).  `roofline.frac` uses SURVEY.md section 8(d)'s per-unit figures (30 / 70 per
# Schwarzschild / Kerr RHS, 55 per RK4 step, 330 per DP5(4) step; for Manko-Novikov the survey gives a
# range, 600-1000, "builder to count": 760).  The builder's own count of the formulas of SURVEY.md
# appendix A/B as written out in csrc/gp_metric.cuh is printed beside it (`frac_builder_model`). ------
F_RHS = {W.SCHWARZSCHILD: 30.0, W.KERR: 70.0, W.MANKO_NOVIKOV: 760.0}
F_STEP = {0: 55.0, 1: 55.0, 2: 330.0}
F_RHS_BUILDER = {W.SCHWARZSCHILD: 40.0, W.KERR: 81.0, W.MANKO_NOVIKOV: 760.0}
F_STEP_BUILDER = {0: 56.0, 1: 57.0, 2: 324.0}
# Counter evidence that one timed run cannot produce (ncu replays kernels; a number printed under ncu is
# never a bench value): hardware-counted FP64 flops / cycle as a fraction of the FMA peak, and DRAM bytes
# per launch, of the SAME kernel build on the SAME workload, each with the profiles/ file it comes from.
# Workloads without a capture report null and say so.
PROFILED = {
    ("headline", "fp64"): {"hw_fp64_frac": 0.512, "traffic": 8.37e7, "source": "profiles/trace_dp54_r02e.md"},
    ("C3", "fp64"): {"hw_fp64_frac": 0.500, "traffic": 1.334e8, "source": "profiles/kernels_r02g.md"},
    ("headline_rk4", "fp64"): {"hw_fp64_frac": 0.523, "traffic": 8.26e7, "source": "profiles/kernels_r02g.md"},
    ("headline_rk4", "fp32"): {"hw_fp64_frac": None, "hw_fp32_frac": 0.386, "traffic": 8.12e7,
                               "source": "profiles/kernels_r02g.md"},
    ("headline_rk4", "mixed"): {"hw_fp64_frac": 0.102, "hw_fp32_frac": 0.246, "traffic": 8.12e7,
                                "source": "profiles/kernels_r02g.md"},
    ("C5a", "fp32"): {"hw_fp64_frac": None, "hw_fp32_frac": 0.417, "traffic": 2.12e9,
                      "source": "profiles/kernels_r02g.md"},
}
# captures taken at an overridden image size (--side): the Manko-Novikov configs at a size ncu can replay
PROFILED_AT_SIDE = {
    ("C4", "fp64", 512): {"hw_fp64_frac": 0.252, "traffic": 5.07e5,
                          "source": "profiles/trace_dp54_mn_r02.md (addendum r02b; 17 of 32 lanes live at this size)"},
}
# nominal FP64 FMA peak: 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz
FP64_LANES_PER_SM = 64
FP32_LANES_PER_SM = 128


def _args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="headline")
    ap.add_argument("--side", type=int, default=0,
                    help="override the image size of the workload (side x side pixels); for profiling the "
                         "Manko-Novikov configs at a size ncu can replay")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=12.0,
                    help="target oracle time for the cpu_baseline sample")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "mixed"],
                    help="fp32: the single-precision variant (fixed-step RK4 workloads only); mixed: FP32 "
                         "equations with an FP64 state (adaptive workloads run at rtol = atol = 1e-7)")
    ap.add_argument("--stage", default="trace", choices=["trace", "shade"],
                    help="shade: time the image-formation kernel gp_shade on the records of a 2048^2 frame")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one frame per rank; strong = ONE frame split cyclically over the ranks "
                         "(gp_workloads.shard, DESIGN.md section 8)")
    ap.add_argument("--back-to-back", type=int, default=8,
                    help="images of the extra back-to-back measurement on two streams (0 = skip)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


# ---- clocks during the timed region (B200_PROFILING.md recipe) ------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln)

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(self.NAMES, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def alg_flops(w, attempts, n_rhs, builder=False):
    """Algorithmic FP64 flops of a trace from its step and RHS counts."""
    fr, fs = (F_RHS_BUILDER, F_STEP_BUILDER) if builder else (F_RHS, F_STEP)
    return fr[w["metric"]["id"]] * float(n_rhs) + fs[w["cfg"]["scheme"]] * float(attempts)


def config_of(w, n_gpus, extra=None):
    cam, cfg = w["camera"], w["cfg"]
    c = {"workload": w["name"],
         "metric_id": {0: "schwarzschild", 1: "kerr", 2: "manko_novikov"}[w["metric"]["id"]],
         "a": w["metric"]["a"], "q": w["metric"]["q"],
         "image": f"{cam['width']}x{cam['height']}x{cam['supersample']}^2",
         "rays_per_step_per_gpu": W.n_rays(w),
         "scheme": {0: "rk4_fixed", 1: "rk4_h_rel", 2: "dp54_adaptive"}[cfg["scheme"]],
         "rtol": cfg["rtol"], "r_obs": cam["r_obs"],
         "parallelism": f"frames{n_gpus}" if n_gpus > 1 else "single",
         "l2": "each step writes 128 MiB of records (> 126 MB L2); the path reads no input arrays"}
    if extra:
        c.update(extra)
    return c


# ---- the oracle, timed (cpu_baseline leg and --impl reference) --------------------------------------
def oracle_sample(w, seconds, single_thread_seconds=0.0):
    """Time the oracle on a scattered subsample of the workload sized for about `seconds`."""
    from oracle import oracle as O
    total = W.n_rays(w)
    probe = min(total, 4096)
    stride = max(1, total // probe) | 1
    b, c, s = W.ray_selection(w, 1, probe, stride)
    # all host cores, also under torchrun (which exports OMP_NUM_THREADS=1)
    cores = os.cpu_count() or 1
    t0 = time.perf_counter()
    _, used = O.trace(w, b, c, s, n_threads=cores)
    rate = c / max(time.perf_counter() - t0, 1e-6)
    count = int(min(total, max(probe, rate * seconds)))
    stride = 1 if count >= total else (-(-total // count)) | 1   # odd stride: the sample scatters over the image
    b, c, s = W.ray_selection(w, 0, None, stride)
    t0 = time.perf_counter()
    rec, used = O.trace(w, b, c, s, n_threads=cores)
    dt = time.perf_counter() - t0
    out = {"value": c / dt, "unit": "geodesics/s", "cores": int(used), "kind": "oracle",
           "sample": f"{c} rays of {w['name']} (ray stride {s} from ray {b}), {dt:.2f} s wall, "
                     f"OpenMP dynamic over rays, g++ -O2 -ffp-contract=off",
           "rhs_evals_per_s": float(rec["n_rhs"].sum()) / dt, "seconds": dt, "rays": c}
    if single_thread_seconds > 0:
        # "also the single-thread rate" — a smaller sample of the same kind, one thread
        c1 = int(max(256, min(c, out["value"] / max(1, used) * single_thread_seconds)))
        b1, c1, s1 = W.ray_selection(w, 0, c1, (-(-total // c1)) | 1)
        t0 = time.perf_counter()
        O.trace(w, b1, c1, s1, n_threads=1)
        dt1 = time.perf_counter() - t0
        out["single_thread"] = {"value": c1 / dt1, "unit": "geodesics/s",
                                "sample": f"{c1} rays (stride {s1}), {dt1:.2f} s wall, 1 thread"}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = W.workload(args.workload)
    per_step = max(1.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(w, per_step / 4)
    rates, cpu, t_all = [], None, 0.0
    rays = 0
    for _ in range(args.steps):
        cpu = oracle_sample(w, per_step)
        rays += cpu["rays"]
        t_all += cpu["seconds"]
    value = rays / t_all
    cpu = {k: cpu[k] for k in ("unit", "cores", "kind", "sample")}
    cpu["value"] = value
    print(json.dumps({
        "impl": "reference", "metric": "geodesics/sec (1024^2 Kerr a=0.9, FP64)", "value": value,
        "unit": "geodesics/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_all / max(1, args.steps), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_of(w, 1, {"note": "each step = a bounded scattered sample of the image"}),
        "cpu_baseline": cpu,
        "e2e": {"value": value, "unit": "geodesics/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ---- the CUDA path ---------------------------------------------------------------------------------
def run_b200(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_2310_15183_b200 as gp  # raises if libgp.so cannot be built/loaded: no fallback

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA library is the product, there is no CPU path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # Rays are independent, so there is no exchange step.  weak: every rank traces
    # its own frame of the workload (its own jitter seed).  strong: ONE frame, rank g takes the rays
    # g, g + G, g + 2G, ... (gp_workloads.shard: cost per ray varies strongly over the image, cyclic
    # interleave balances it); each rank runs its own work counter into its own buffers.
    w = W.workload(args.workload, **(dict(width=args.side, height=args.side) if args.side else {}))
    strong = args.scaling == "strong" and world > 1
    if not strong:
        w["camera"]["jitter_seed"] = int(w["camera"].get("jitter_seed", 0)) + rank
    mixed = args.precision == "mixed"
    fp32 = args.precision == "fp32" or mixed        # which roofline: the equations run on the FP32 lanes
    if args.precision == "fp32":
        if w["cfg"]["scheme"] == 2:
            raise SystemExit("bench.py: --precision fp32 exists for the fixed-step RK4 workloads only")
        w["cfg"]["precision"] = 1
    if mixed:
        w["cfg"]["precision"] = 2
        if w["cfg"]["scheme"] == 2:
            w["cfg"].update(rtol=1e-7, atol=1e-7)   # gp.h: the floor of the mixed adaptive variant
    n_frame = W.n_rays(w)
    sel = W.shard(w, rank, world) if strong else W.ray_selection(w)
    n = sel[1]                      # rays this rank traces per step
    mid = w["metric"]["id"]
    ms, cs, gs = gp.api.metric_struct(w["metric"]), gp.api.camera_struct(w["camera"], *sel), gp.api.cfg_struct(w["cfg"])
    disk_on = gs.max_crossings > 0
    rays = torch.empty(n * 128, dtype=torch.uint8, device=dev)
    disk = torch.empty(n * 48, dtype=torch.uint8, device=dev) if disk_on else None
    counters = torch.zeros(64, dtype=torch.uint8, device=dev)
    scratch = torch.zeros(8, dtype=torch.uint8, device=dev)
    stream = torch.cuda.Stream(device=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def step():
        gp.gp_trace(mid, ms, cs, gs, rays, disk, counters, stream)

    def probe_peak():
        """DFMA-chain probe (gp_probe_fp64_fma) -> TFLOP/s at the clocks of this moment."""
        best = 0.0
        with torch.cuda.stream(stream):
            gp.gp_probe_fp64_fma(2000, scratch, stream)
            for _ in range(3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                fl = gp.gp_probe_fp64_fma(40000, scratch, stream)
                e1.record(stream)
                e1.synchronize()
                best = max(best, fl / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        return best

    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            step()
    barrier()
    peak_probe = probe_peak()

    # ---- device-resident timed region: exactly K steps, CUDA events on the launching stream ----
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    barrier()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with torch.cuda.stream(stream):
        ev[0].record(stream)
        for i in range(args.steps):
            step()
            ev[i + 1].record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = ev[0].elapsed_time(ev[-1])
    per_launch_ms = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps))
    cnt = counters.cpu().numpy().view("<u8")
    assert int(cnt[1]) == n, "every ray must finish exactly once"
    attempts, n_rhs = int(cnt[2]), int(cnt[3])
    tmax = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    total_ms_max = float(tmax.item())

    # ---- back to back ("also time 8 back-to-back images"): the same frame traced B
    # times on two streams into two sets of buffers, so that the end-of-image tail of one launch (lanes
    # going idle once the work counter is exhausted, `tail` below) overlaps the start of the next.
    # Reported beside `value`, which stays the one-launch-at-a-time figure. ----
    b2b = None
    if args.back_to_back >= 2 and world == 1:
        streams = [stream, torch.cuda.Stream(device=dev)]
        bufs = [(rays, disk, counters),
                (torch.empty_like(rays), torch.empty_like(disk) if disk_on else None, torch.zeros_like(counters))]
        torch.cuda.synchronize(dev)
        for rep in range(2):            # first pass warms the second stream
            t_ev0, t_ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t_ev0.record(streams[0])
            streams[1].wait_event(t_ev0)
            for i in range(args.back_to_back):
                r_, d_, c_ = bufs[i % 2]
                gp.gp_trace(mid, ms, cs, gs, r_, d_, c_, streams[i % 2])
            streams[0].wait_stream(streams[1])
            t_ev1.record(streams[0])
            t_ev1.synchronize()
            b2b_ms = t_ev0.elapsed_time(t_ev1) / args.back_to_back
        for _, _, c_ in bufs:
            assert int(c_.cpu().numpy().view("<u8")[1]) == n
        b2b = {"images": args.back_to_back, "streams": 2, "ms_per_image": b2b_ms,
               "geodesics_per_s": n / (b2b_ms * 1e-3)}

    # ---- end to end: gp_trace_host into pinned host buffers (alloc + kernel + D2H + sync) ----
    e2e = None
    if not args.no_e2e:
        h_rays = torch.empty(n * 128, dtype=torch.uint8, pin_memory=True).numpy().view(gp.api.RAY_DTYPE)
        h_disk = (torch.empty(n * 48, dtype=torch.uint8, pin_memory=True).numpy().view(gp.api.DISK_DTYPE)
                  if disk_on else None)
        h_cnt = np.zeros(8, dtype=np.uint64)
        for _ in range(2):
            gp.gp_trace_host(mid, ms, cs, gs, h_rays, h_disk, h_cnt, stream)
        barrier()
        k_e2e = max(3, min(args.steps, 10))
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            gp.gp_trace_host(mid, ms, cs, gs, h_rays, h_disk, h_cnt, stream)  # synchronises the stream
        torch.cuda.synchronize(dev)
        dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(dt, op=dist.ReduceOp.MAX)
        assert int(h_cnt[1]) == n and int((h_rays["status"] <= 4).sum()) == n
        e2e = {"value": (n_frame if strong else world * n) * k_e2e / float(dt.item()), "unit": "geodesics/s",
               "h2d_bytes_per_step": 24 + 120 + 112,  # the three parameter structs, as kernel arguments
               "d2h_bytes_per_step": n * 128 + (n * 48 if disk_on else 0) + 64,
               "steps": k_e2e, "call": "gp_trace_host (pinned host records, stream sync inside)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    sec = total_ms_max * 1e-3
    n_job = n_frame if strong else world * n          # rays all ranks trace per step
    value = n_job * args.steps / sec
    kern_ms = sum(per_launch_ms) / len(per_launch_ms)
    flops = alg_flops(w, attempts, n_rhs)
    achieved = flops / (kern_ms * 1e-3) / 1e12
    achieved_builder = alg_flops(w, attempts, n_rhs, builder=True) / (kern_ms * 1e-3) / 1e12
    none = {"hw_fp64_frac": None, "traffic": None,
            "source": "no ncu capture of this workload / precision / size under profiles/"}
    prof = (PROFILED_AT_SIDE.get((args.workload, args.precision, args.side), none) if args.side
            else PROFILED.get((args.workload, args.precision), none))
    props = torch.cuda.get_device_properties(dev)
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    lanes = FP32_LANES_PER_SM if fp32 else FP64_LANES_PER_SM
    peak_nominal = props.multi_processor_count * lanes * 2 * sm_max * 1e6 / 1e12
    out = {
        "metric": "geodesics/sec (1024^2 Kerr a=0.9, FP64)" if args.workload == "headline"
                  else f"geodesics/sec ({args.workload})",
        "value": value, "unit": "geodesics/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": total_ms_max / args.steps,
        # per-launch CUDA-event times of this rank over the timed region (best and median)
        "ms_per_step_best": per_launch_ms[0], "ms_per_step_median": per_launch_ms[len(per_launch_ms) // 2],
        "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None,
        "dtype": "f32 equations + f64 state" if mixed else ("f32" if fp32 else "f64"),
        "data": "synthetic",
        "config": config_of(w, world, {"parallelism": f"cyclic_shards{world}", "rays_per_step_per_gpu": n} if strong else None),
        "rhs_evals_per_s": world * n_rhs * args.steps / sec,      # rank 0's count x ranks
        "steps_per_ray": attempts / n, "rhs_per_ray": n_rhs / n,
        "roofline": {"bound": "alu", "kernel": "trace_dp54" if gs.scheme == 2 else "trace_rk4",
                     "achieved": achieved, "peak": peak_nominal, "unit": "TFLOP/s",
                     "frac": achieved / peak_nominal,
                     "flop_model": f"SURVEY.md 8(d): {F_RHS[mid]:.0f}/RHS + {F_STEP[gs.scheme]:.0f}/step",
                     "frac_builder_model": achieved_builder / peak_nominal,
                     "builder_model": f"{F_RHS_BUILDER[mid]:.0f}/RHS + {F_STEP_BUILDER[gs.scheme]:.0f}/step (DESIGN.md 6.2)",
                     # not measurable inside a timed run: from the ncu --set full capture named in `profile`
                     # (dram__bytes_read.sum + dram__bytes_write.sum per launch; (2 DFMA + DMUL + DADD) / cycle
                     # over 148 SMs x 128 flop / cycle)
                     "traffic": prof["traffic"], "hw_fp64_frac": prof["hw_fp64_frac"],
                     "hw_fp32_frac": prof.get("hw_fp32_frac"), "profile": prof["source"],
                     "peak_kind": f"nominal {'FP32' if fp32 else 'FP64'} FMA: {props.multi_processor_count} SMs x "
                                  f"{lanes} lanes x 2 x {sm_max:.0f} MHz",
                     "peak_probe": None if fp32 else peak_probe,
                     "frac_of_probe": None if fp32 else (achieved / peak_probe if peak_probe else None),
                     "probe_kind": "gp_probe_fp64_fma: register-resident DFMA chains, same process",
                     "alg_flops_per_launch": flops, "kernel_ms": kern_ms},
        "clocks": clocks, "gpu_launches": args.steps,
        # end-of-image tail of the persistent kernel, from the device time stamps of the last launch
        # (gp.h counters[4..7]): steady-state rate = 99 % of the rays / time until they had finished
        "tail": {"kernel_ms": (int(cnt[7]) - int(cnt[4])) * 1e-6,
                 "t99_ms": (int(cnt[5]) - int(cnt[4])) * 1e-6 if int(cnt[5]) else None,
                 "steady_geodesics_per_s": ((n - n // 100) / ((int(cnt[5]) - int(cnt[4])) * 1e-9)
                                            if int(cnt[5]) > int(cnt[4]) else None)},
    }
    if b2b:
        out["back_to_back"] = b2b
    if e2e:
        out["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        cpu = oracle_sample(w, args.cpu_seconds, single_thread_seconds=3.0)
        out["cpu_baseline"] = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "rhs_evals_per_s",
                                                   "single_thread")}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


# ---- image formation (gp_shade): an HBM-bound step, reported against the measured copy bandwidth ----
def run_shade(args):
    import numpy as np
    import torch
    import paper_2310_15183_b200 as gp
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device")
    torch.cuda.set_device(0)
    side = 2048                                   # 512 MiB of records: four times the L2
    w = W.workload(args.workload, width=side, height=side)
    n = W.n_rays(w)
    rays = torch.empty(n * 128, dtype=torch.uint8, device="cuda")
    counters = torch.zeros(64, dtype=torch.uint8, device="cuda")
    out = torch.empty(n * 4, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.Stream()
    gp.gp_trace(w["metric"]["id"], gp.api.metric_struct(w["metric"]), gp.api.camera_struct(w["camera"]),
                gp.api.cfg_struct(w["cfg"]), rays, None, counters, stream)
    cfg = gp.api.shade_struct(dict(width=side, height=side, mode=1, tex_width=4096, tex_height=2048, tex_seed=1))
    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            gp.gp_shade(cfg, rays, None, out, stream)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.3)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with torch.cuda.stream(stream):
        ev[0].record(stream)
        for i in range(args.steps):
            gp.gp_shade(cfg, rays, None, out, stream)
            ev[i + 1].record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = ev[0].elapsed_time(ev[-1]) / args.steps
    # end to end: pinned host records in, pinned host image out
    h_rays = torch.empty(n * 128, dtype=torch.uint8, pin_memory=True)
    h_rays.copy_(rays)
    h_out = torch.empty(n * 4, dtype=torch.uint8, pin_memory=True)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    k_e2e = 3
    with torch.cuda.stream(stream):
        for _ in range(k_e2e):
            rays.copy_(h_rays, non_blocking=True)
            gp.gp_shade(cfg, rays, None, out, stream)
            h_out.copy_(out, non_blocking=True)
    stream.synchronize()
    dt = (time.perf_counter() - t0) / k_e2e
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peak, kind = float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (copy bandwidth, burst)"
    except (OSError, KeyError, ValueError):
        peak, kind = 6650.0, "of fallback (B200_PROFILING.md: 6.65 TB/s)"
    alg_bytes = n * (28 + 4)          # t, theta, phi, status read; one RGBA8 pixel written
    achieved = alg_bytes / (ms * 1e-3) / 1e9
    print(json.dumps({
        "metric": f"pixels/s (image formation, {side}^2 {args.workload} records, bilinear texture)",
        "value": n / (ms * 1e-3), "unit": "pixels/s", "n_gpus": 1, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload} at {side}x{side}", "stage": "shade", "mode": "texture 4096x2048",
                   "l2": "512 MiB of records read per step (> 126 MB L2)"},
        "roofline": {"bound": "hbm", "kernel": "k_shade", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak,
                     # dram__bytes_read.sum + dram__bytes_write.sum of one launch (profiles/kernels_r01d.md)
                     "traffic": 2.861e8, "peak_kind": kind,
                     "alg_bytes_per_launch": alg_bytes,
                     "note": "the reader needs 28 bytes per record, all in its first 64-byte half (ld with an "
                             "L2::64B hint: 268 MB read per launch, was 537 MB); the kernel is then bound by its six "
                             "IEEE FP64 divisions per sub-ray, not by HBM (profiles/kernels_r01d.md)"},
        "clocks": clocks, "gpu_launches": args.steps,
        "e2e": {"value": n / dt, "unit": "pixels/s", "h2d_bytes_per_step": n * 128, "d2h_bytes_per_step": n * 4}}))


if __name__ == "__main__":
    a = _args()
    if a.impl == "reference":
        run_reference(a)
    elif a.stage == "shade":
        run_shade(a)
    else:
        run_b200(a)
