"""bench.py - ms per second-order DLR step (Algorithm 2) and achieved HBM GB/s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

Workload at N=1: BASELINE.json configs[2] ("config 3": two-stream 64^3 x 64^3, r = 10, fp64, tau = 0.05), the shape
the metric is quoted on.  A "step" is one pass of the whole hot path (dlr_step).  N > 1: independent replicas, one
per rank, no collective on the data path ("replicas only") -> weak scaling, value = ms per
step (time-like: max over ranks).  --impl reference times the NumPy oracle on the host cores (rank 0 only).
Prints ONE JSON line.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

def metric_name(cfg):
    return f"ms per 2nd-order DLR step ({cfg['n_x']}^3x{cfg['n_v']}^3, r={cfg['r']}, fp64)"


# fp64 vector peak of the B200 (no such entry in MEASURED_PEAKS.json / B200_PROFILING.md): 148 SMs x 4 sub-partitions x 16
# fp64 lanes x 2 flop x 1.965 GHz = 37.2 TFLOP/s; a DFMA-only kernel measured 36.8 on this pool (profiles/r02_peaks.md).
# DMMA (mma.sync.m8n8k4.f64) measured 37.2: the fp64 tensor path has the same peak as the vector path.
FP64_TFLOPS = 36.8


def clocks_sampler(stop, out, dev):
    q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    while not stop.is_set():
        try:
            r = subprocess.run(["nvidia-smi", f"--id={dev}", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                               capture_output=True, text=True, timeout=5)
            out.append([x.strip() for x in r.stdout.strip().split(",")])
        except Exception:
            pass
        stop.wait(0.1)


def summarize_clocks(samples):
    sm = sorted(int(s[0]) for s in samples if len(s) >= 6 and s[0].isdigit())
    mx = [int(s[1]) for s in samples if len(s) >= 6 and s[1].isdigit()]
    names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    reasons = [n for i, n in enumerate(names) if any(len(s) >= 6 and s[2 + i] == "Active" for s in samples)]
    return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p))["hbm_gbs"], "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# kernel families of one step: substring of the launch expression (dlr_set_profiling(ctx, 2)) -> (label, algorithmic
# bytes per launch as (factor passes, field components): B = 8 N r per factor read or write,
# 8 N per field component).  Averages over the launches of a step where K and L flows differ.
# Algorithmic flops per grid point (all r columns) of a launch, (r, log2 n) -> flops: column mixing 2 r^2 per r x r product,
# a 1D real transform 2.5 log2(n) per point and column.
FAMILIES = [
    ("run_sub1", "k_sub1 sub-flow 1 + both basis changes (warp-autonomous units)", 2.0, 0.0,
     lambda r, lg: 4 * r * r + 5 * lg * r),
    ("run_sub2", "k_sub2 sub-flow 2 (warp-autonomous units)", 2.0, 0.0, lambda r, lg: 5 * lg * r + 6 * r),
    ("VD_ETD2", "k_dir<r,3,ETD2> third sub-flow, both ETD2RK stages", 2.0, 2.0,      # E read by 2 of 3 launches
     lambda r, lg: 16 * r * r + 12.5 * lg * r),
    ("VD_ETD1", "k_dir<r,3,ETD1> third sub-flow, exponential Euler", 2.0, 3.0,
     lambda r, lg: 10 * r * r + 7.5 * lg * r),
    ("VD_COEFF1", "k_dir<r,1,COEFF> weighted Gram + Parseval", 1.0, 2.0, lambda r, lg: 4 * r * (r + 1) + 2.5 * lg * r + 2 * r * r),
    ("VD_COEFF2", "k_dir<r,2,COEFF> Parseval", 1.0, 0.0, lambda r, lg: 2.5 * lg * r + 2 * r * r),
    ("VD_COEFF3", "k_dir<r,3,COEFF> Parseval", 1.0, 0.0, lambda r, lg: 2.5 * lg * r + 2 * r * r),
    ("ops->apply", "k_apply CholeskyQR A*R^-1 (+ Gram), bulk-copy pipeline", 2.0, 0.0, lambda r, lg: 2 * r * r + r * (r + 1)),
]


def kernel_breakdown(ctx, tau, cfg, nprof=5):
    """per-launch device times of `nprof` steps (CUDA events after every launch, direct launches on the context's
    stream), grouped into kernel families"""
    import numpy as np
    ctx.set_profiling(2)
    runs = []
    for _ in range(nprof):
        ctx.step(tau)
        runs.append(ctx.phase_times())
    ctx.set_profiling(0)
    names = [n for n, _ in runs[0]]
    ms = np.median(np.array([[t for _, t in r] for r in runs]), axis=0)
    B = 8.0 * (0.5 * (cfg["n_x"] ** 3 + cfg["n_v"] ** 3)) * cfg["r"]     # x and v passes alternate: mean factor size
    EN = 8.0 * cfg["n_x"] ** 3
    fam = {}
    total = float(sum(t for t in ms if t > 0))
    for n, t in zip(names, ms):
        for key, label, nb, ne, fl in FAMILIES:
            if key in n:
                if key == "ops->apply" and t < 0.010:        # the skipped third CholeskyQR stage: a no-op launch
                    break
                npts = 0.5 * (cfg["n_x"] ** 3 + cfg["n_v"] ** 3)
                lg = 0.5 * (math.log2(cfg["n_x"]) + math.log2(cfg["n_v"]))
                f = fam.setdefault(label, {"launches": 0, "ms": 0.0, "bytes": nb * B + ne * EN,
                                           "flops": fl(cfg["r"], lg) * npts})
                f["launches"] += 1
                f["ms"] += float(t)
                break
    out = []
    for label, f in fam.items():
        avg_us = 1e3 * f["ms"] / f["launches"]
        out.append({"kernel": label, "launches_per_step": f["launches"], "avg_us": avg_us,
                    "share_of_step": f["ms"] / total, "algorithmic_bytes_per_launch": f["bytes"],
                    "gbs": f["bytes"] / (avg_us * 1e-6) / 1e9,
                    "algorithmic_flops_per_launch": f["flops"], "tflops": f["flops"] / (avg_us * 1e-6) / 1e12})
    out.sort(key=lambda k: -k["share_of_step"])
    return out


def oracle_leg(cfg, steps, warmup):
    """the oracle as it stands on the host cores, on a bounded sample: `steps` full steps of the SAME workload"""
    import numpy as np
    from oracle import dlr_oracle as O
    from paper_2110_13481_b200 import inputs
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        cores = 1
    gx = O.Grid3((cfg["n_x"],) * 3, (cfg["x_lo"],) * 3, (cfg["x_hi"],) * 3)
    gv = O.Grid3((cfg["n_v"],) * 3, (cfg["v_lo"],) * 3, (cfg["v_hi"],) * 3)
    X, S, V = inputs.initial_factors(cfg)
    for _ in range(warmup):
        X, S, V = O.step_alg2(X, S, V, cfg["tau"], gx, gv)
    t0 = time.perf_counter()
    for _ in range(steps):
        X, S, V = O.step_alg2(X, S, V, cfg["tau"], gx, gv)
    ms = (time.perf_counter() - t0) * 1e3 / max(steps, 1)
    return ms, cores


def oracle_single_thread(cfg):
    """one step of the oracle with the BLAS pool limited to one thread (pocketfft is single-threaded anyway)"""
    try:
        from threadpoolctl import threadpool_limits
    except Exception:
        return None
    with threadpool_limits(limits=1):
        ms, _ = oracle_leg(cfg, 1, 0)
    return ms


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200, help="steps per timed block (K)")
    ap.add_argument("--min-seconds", type=float, default=1.2,
                    help="K-step blocks are repeated (each timed on its own) until this much device time and 5 blocks")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--n-x", type=int, default=0, help="override the x grid of --config (the paper's anisotropic shapes)")
    ap.add_argument("--n-v", type=int, default=0, help="override the v grid of --config")
    ap.add_argument("--rank", type=int, default=0, help="override the rank of --config")
    ap.add_argument("--cpu-steps", type=int, default=1, help="oracle steps timed for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--unconventional", action="store_true",
                    help="time the unconventional integrator (DLR_FLAG_UNCONVENTIONAL, first order) instead of Algorithm 2; "
                         "not the headline metric: use with --no-cpu-baseline")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    from paper_2110_13481_b200 import inputs
    over = {}
    if args.n_x:
        over["n_x"] = args.n_x
    if args.n_v:
        over["n_v"] = args.n_v
    if args.rank:
        over["r"] = args.rank
    cfg = inputs.make_config(args.config, **over)
    workload = (f"BASELINE.json configs[{args.config - 1}]: {cfg['problem']} {cfg['n_x']}^3x{cfg['n_v']}^3, r={cfg['r']}, "
                f"tau={cfg['tau']}, Algorithm 2")
    if args.unconventional:
        workload = workload.replace("Algorithm 2", "unconventional integrator (reference [4] of the paper)")
    config = {"workload": workload, "n": cfg["n"], "rank": cfg["r"], "tau": cfg["tau"], "parallelism": f"replicas x{args.gpus}",
              "l2": (f"working set {6 * 8 * max(cfg['n_x'], cfg['n_v']) ** 3 * cfg['r'] / 1e9:.2f} GB of factors and work buffers; "
                     "126 MB L2: no explicit flush, but at 64^3 a single 21 MB factor is L2-resident between consecutive passes "
                     "(configs 4 and 5 are the HBM-resident cases, BASELINE.md)")}
    METRIC = metric_name(cfg)

    if args.impl == "reference":
        if rank != 0:
            return
        steps = max(1, min(args.steps, 2))
        ms, cores = oracle_leg(cfg, steps, min(args.warmup, 1))
        print(json.dumps({
            "impl": "reference", "metric": METRIC, "value": ms, "unit": "ms/step", "n_gpus": args.gpus, "steps": steps,
            "warmup": min(args.warmup, 1), "ms_per_step": ms, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config,
            "cpu_baseline": {"value": ms, "unit": "ms/step", "cores": cores, "kind": "oracle",
                             "sample": f"{steps} full step(s) of the same workload (NumPy oracle, pocketfft single-threaded)"},
            "e2e": {"value": ms, "unit": "ms/step", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2110_13481_b200 import dlr, replicas
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the hot path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    X, S, V = inputs.initial_factors(replicas.replica_cfg(cfg, rank))
    stream = torch.cuda.Stream(device=dev)
    if args.unconventional:
        METRIC = METRIC.replace("2nd-order DLR step", "unconventional-integrator step (first order)")
        X, S, V = inputs.weighted_start(replicas.replica_cfg(cfg, rank))
    dcfg = (dlr.config_from_inputs(cfg, order=1, flags=dlr.FLAG_UNCONVENTIONAL) if args.unconventional
            else dlr.config_from_inputs(cfg))
    ctx = dlr.Dlr(dcfg, device=dev, stream=stream)
    Xd, Sd, Vd = (torch.from_numpy(np.ascontiguousarray(a.T)).to(dev) for a in (X, S, V))   # column-major on device
    tau = cfg["tau"]

    # ---- device-resident timing: K steps, CUDA events on the launching stream
    ctx.set_initial(Xd, Sd, Vd)
    for _ in range(max(args.warmup, 3)):
        ctx.step(tau)
    barrier()
    samples, stop = [], threading.Event()
    th = threading.Thread(target=clocks_sampler, args=(stop, samples, local_rank))
    th.start()
    # K-step blocks, each between its own pair of events on the launching stream; repeated until >= --min-seconds of device
    # time and >= 5 blocks so that the clocks are sampled under sustained load.  value = median block.
    barrier()
    blocks = []
    while (sum(blocks) < args.min_seconds * 1e3 or len(blocks) < 5) and len(blocks) < 200:
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            ev0.record(stream)
            for _ in range(args.steps):
                ctx.step(tau)
            ev1.record(stream)
        barrier()
        blocks.append(ev0.elapsed_time(ev1))
    per_step = sorted(b / args.steps for b in blocks)
    ms_step = per_step[len(per_step) // 2]
    stop.set()
    th.join()
    mom = ctx.moments()
    launches = ctx.launches_per_step()
    bytes_step = ctx.bytes_per_step()
    kernels = kernel_breakdown(ctx, tau, cfg)

    # ---- end to end through the public API with HOST buffers: set_initial(host) + K steps + moments() each
    # step (device->host read of the diagnostics) + get_factors(host) at the end, all inside the timed region
    Xp, Sp, Vp = (torch.from_numpy(np.ascontiguousarray(a.T)).pin_memory() for a in (X, S, V))
    Xo, So, Vo = (torch.empty_like(t).pin_memory() for t in (Xp, Sp, Vp))      # pinned destination of get_factors
    e2e_steps = max(1, min(args.steps, 10))
    barrier()
    t0 = time.perf_counter()
    ctx.set_initial(Xp, Sp, Vp)
    for _ in range(e2e_steps):
        ctx.step(tau)
        ctx.moments()
    ctx.get_factors(out=(Xo, So, Vo))
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
    fac_bytes = (X.nbytes + S.nbytes + V.nbytes)
    h2d = fac_bytes / e2e_steps
    d2h = fac_bytes / e2e_steps + 80

    ms_step, e2e_ms = replicas.max_over_ranks([ms_step, e2e_ms], dev, world)

    if rank == 0:
        peak, peak_src = measured_peak()
        achieved = bytes_step / (ms_step * 1e-3) / 1e9
        top = kernels[0]
        traffic = None
        tpath = os.path.join(ROOT, "profiles", "r02_traffic.json")
        if os.path.exists(tpath):
            traffic = json.load(open(tpath)).get(top["kernel"].split(" ")[0])
        # which roofline binds a kernel: the larger of its two floors, algorithmic bytes / HBM peak and algorithmic
        # fp64 flops / fp64 peak (plain ALUs: the fp64 tensor path has the same peak on B200)
        for k in kernels:
            t_hbm = k["algorithmic_bytes_per_launch"] / (peak * 1e9)
            t_alu = k["algorithmic_flops_per_launch"] / (FP64_TFLOPS * 1e12)
            k["bound"] = "alu" if t_alu > t_hbm else "hbm"
            k["frac"] = max(t_hbm, t_alu) / (k["avg_us"] * 1e-6)
            k["frac_hbm"], k["frac_alu"] = k["gbs"] / peak, k["tflops"] / FP64_TFLOPS
        flops_step = sum(k["algorithmic_flops_per_launch"] * k["launches_per_step"] for k in kernels)
        alu = top["bound"] == "alu"
        roofline = {
            "bound": top["bound"], "kernel": top["kernel"],
            "achieved": top["tflops"] if alu else top["gbs"], "peak": FP64_TFLOPS if alu else peak,
            "unit": "TFLOP/s" if alu else "GB/s", "frac": top["frac"], "traffic": traffic,
            "peak_source": ("fp64 vector peak derived in DESIGN.md section 6: 148 SMs x 64 fp64 lanes x 2 x 1.965 GHz = 37.2 "
                            "TFLOP/s, a DFMA-only kernel measured 36.8 on this pool (profiles/r02_peaks.md); HBM: " + peak_src)
                           if alu else peak_src,
            "algorithmic_bytes_per_launch": top["algorithmic_bytes_per_launch"],
            "algorithmic_flops_per_launch": top["algorithmic_flops_per_launch"], "avg_launch_us": top["avg_us"],
            "launches_per_step": top["launches_per_step"], "share_of_step": top["share_of_step"],
            "hbm": {"achieved": top["gbs"], "peak": peak, "unit": "GB/s", "frac": top["gbs"] / peak, "peak_source": peak_src},
            "alu": {"achieved": top["tflops"], "peak": FP64_TFLOPS, "unit": "TFLOP/s", "frac": top["tflops"] / FP64_TFLOPS},
            "note": "dominant kernel family of the step by device time; duration = CUDA events after every launch on "
                    "the context's stream (dlr_set_profiling(ctx, 2), 5 steps, median) right after the timed region; "
                    "traffic = DRAM bytes per launch from the ncu --set full capture of this build in profiles/ (cold "
                    "cache). bound = the larger of the kernel's two floors (algorithmic bytes / measured HBM copy peak, "
                    "algorithmic fp64 flops / fp64 peak): the third sub-flow has 13 flop per byte against a machine balance "
                    "of 5.6, so the fp64 ALUs bound it; both fractions are in hbm/alu. As measured (profiles/) no pass kernel "
                    "is HBM-bound at this shape (DRAM traffic = algorithmic bytes, the 21 MB factor is L2-resident) and none "
                    "reaches its ALU floor: they are latency-, barrier- and instruction-fetch-bound (warps active ~22 %, "
                    "issue slots ~33 %, fp64 pipe ~30 %)",
            "step": {"algorithmic_bytes_per_step": bytes_step, "achieved": achieved, "frac": achieved / peak,
                     "alu_tflops": flops_step / (ms_step * 1e-3) / 1e12,
                     "alu_frac": flops_step / (ms_step * 1e-3) / 1e12 / FP64_TFLOPS,
                     "what": "all factor-sized passes of one step (DESIGN.md section 6) / CUDA-event time of the step; "
                             "alu_*: the algorithmic fp64 flops of the pass kernels of one step / the same time"},
            "kernels": kernels,
        }
        out = {
            "metric": METRIC, "value": ms_step, "unit": "ms/step", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config,
            "paper_context": "30.6 ms/step on an A100 at this shape (Table 4, PAPER.md:549; tau=0.01, the paper's own "
                             "two-stream f0): another machine and initial value, context only",
            "clocks": summarize_clocks(samples),
            "e2e": {"value": e2e_ms, "unit": "ms/step", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "what": f"set_initial(pinned host)+{e2e_steps}x(dlr_step+dlr_moments)+get_factors(pinned host), per step"},
            "timed_blocks": {"blocks": len(blocks), "steps_per_block": args.steps, "device_seconds": sum(blocks) / 1e3,
                             "median": ms_step, "min": per_step[0], "max": per_step[-1]},
            "gpu_launches": launches * args.steps,
            "launches_per_step": launches,
            "roofline": roofline,
            "final_state": {"mass": mom["mass"], "electric_energy": mom["electric_energy"],
                            "qr_fallbacks": mom["qr_fallbacks"], "nonfinite": mom["nonfinite"]},
        }
        if world == 1 and not args.no_cpu_baseline:
            cms, cores = oracle_leg(cfg, args.cpu_steps, 0)
            out["cpu_baseline"] = {"value": cms, "unit": "ms/step", "cores": cores, "kind": "oracle", "cpu": cpu_model(),
                                   "single_thread_value": oracle_single_thread(cfg),
                                   "sample": f"{args.cpu_steps} full step(s) of the same workload on the host "
                                             "(NumPy oracle; pocketfft single-threaded, BLAS threads = cores)"}
        print(json.dumps(out))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
