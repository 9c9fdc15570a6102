"""bench.py — throughput of the photon-geodesic hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl gray|reference] [--log2n L] ...

Workload (config.workload): BASELINE config C4, realistic case — 2^L photons per GPU (default L = 30), Kerr a = 0.7,
i = 45 deg, pixels drawn by the seeded counter-based generator over [-15 M, 15 M]^2 at r_obs = 1000 M,
RK4 with the paper's eq. (2) step rule (h = 1/32), termination (capture at 1.01 r_h, escape at
1.01 r_obs, cap 20000 steps) and lane refill (in-register compaction).  One "step" of the benchmark is
one pass of the whole hot path over the batch: gray_init_rays_random -> gray_integrate -> gray_classify
(status histogram read back to the host).  `value` = photon-steps (RK4 steps that advanced a live
photon, counted by the kernel) per second over all GPUs.

--impl reference times the CPU oracle (oracle/, plain C++ fp64) on a bounded strided sample of the same
workload on the host cores; it is a deliberately plain program, not a tuned competitor.
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

# Algorithmic work per photon-step = the oracle's operation tally (oracle.op_tally; add, sub, mul, div,
# sqrt, sin, cos each count 1), asserted equal to these constants by tests/test_bench_constants.py.
FLOPS_PER_PHOTON_STEP = {"rel": 777, "eq2": 787}
# FP32 CUDA-core peak the integrator is bound by: 148 SMs x 128 lanes x 2 (FMA) x
# 1.965 GHz (clocks.max.sm); FP64: 64 lanes per SM.
PEAK_TFLOPS = {"f32": 148 * 128 * 2 * 1.965e9 / 1e12, "f64": 148 * 64 * 2 * 1.965e9 / 1e12}
# dram__bytes_read.sum + dram__bytes_write.sum of one gray_integrate launch of the default workload (2^30 photons,
# fp32) from the committed ncu capture profiles/r01_integrate_f2_dram_2p30.csv: 40.217 GB + 39.874 GB, per photon
NCU_DRAM_BYTES_PER_PHOTON = 74.59
# FP32 operations the packed kernel EXECUTES per photon-step (FMA = 2), from the instruction counts of the committed
# ncu capture (profiles/r01_README.md: FFMA2 166.4, FMUL2 179.4, FADD2 51.1 per warp per step of its 64 photons, plus
# scalar FADD): fewer than the oracle's tally because the kernel contracts the Christoffel sums analytically
NCU_EXECUTED_FLOPS_PER_PHOTON_STEP = 563


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="gray", choices=["gray", "reference"])
    ap.add_argument("--log2n", type=int, default=30, help="photons per GPU = 2^log2n (default: the largest size of BASELINE config C4, "
                    "the north star's 2^30; lowered, and said so in config.workload, if the device lacks the 40 GB it needs)")
    ap.add_argument("--prec", default="f32", choices=["f32", "f64"])
    ap.add_argument("--rule", default="eq2", choices=["eq2", "rel"])
    ap.add_argument("--case", default="realistic", choices=["realistic", "peak", "projection"],
                    help="projection = the paper's first benchmark (P:130-140, Fig. 4): run time of the grid projection "
                         "onto the equatorial plane (a = 0.95, i = 60 deg) against the number of rays")
    ap.add_argument("--schedule", default="refill", choices=["refill", "static"])
    ap.add_argument("--refill-interval", type=int, default=0)
    ap.add_argument("--photons-per-thread", type=int, default=0, help="0 = library default (2 for f32: packed FFMA2), 1, 2")
    ap.add_argument("--system", default="full", choices=["full", "reduced"], help="full = the 8 second-order equations of the north star; reduced = E, L_z eliminate k^t, k^phi")
    ap.add_argument("--xi-eps", type=float, default=0.0, help="epsilon of the paper's xi monitor (P:107); 0 = off")
    ap.add_argument("--e2e-log2n", type=int, default=-1, help="photons per GPU of the host-buffer run (default min(log2n, 26))")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--dist-backend", default="nccl", help="torch.distributed backend of the N > 1 run (the data path has no "
                    "collective; only the timing / counter reduction uses it)")
    ap.add_argument("--share-gpu", action="store_true", help="testing only: all ranks on cuda:0 (use with --dist-backend gloo)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-log2n", type=int, default=18, help="--impl reference: photons of the strided sample per step")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.lines, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, smmax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, line in self.lines:
            if not (t0 <= t <= t1 + 0.25):
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0]))
                smmax = float(f[1])
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smmax, "reasons": sorted(reasons),
                "samples": len(sm)}


def workload_config(args, world):
    from paper_1303_5057_b200 import workloads as wl
    c4 = wl.C4
    return {"workload": f"C4-{args.case}: 2^{args.log2n} photons/GPU, Kerr a={c4['a']}, i={c4['inc_deg']} deg, seeded random "
                        f"pixels over +-{c4['half_width']} M at r_obs={wl.R_OBS:.0f} M, RK4 h=1/32, rule={args.rule}",
            "photons_per_gpu": 2 ** args.log2n, "photons_total": world * 2 ** args.log2n, "precision": args.prec,
            "step_rule": args.rule, "case": args.case, "schedule": args.schedule, "xi_epsilon": args.xi_eps, "system": args.system, "max_steps": wl.MAX_STEPS if args.case == "realistic" else c4["peak_steps"],
            "seed": c4["seed"], "parallelism": f"photon-range sharding x{world}, no collective on the data path",
            "l2": "state (37 B/photon) far larger than the 126 MB L2; no flush needed"}


def oracle_sample(args, log2_sample, threads):
    """Time the oracle on a strided sample of the workload.  Returns (photon_steps, seconds)."""
    import numpy as np

    import oracle as o
    from paper_1303_5057_b200 import workloads as wl
    c4 = wl.C4
    n, m = 2 ** args.log2n, 2 ** min(log2_sample, args.log2n)
    idx = (np.arange(m, dtype=np.uint64) * np.uint64(n // m))
    rule = o.STEP_EQ2 if args.rule == "eq2" else o.STEP_REL
    max_steps = wl.MAX_STEPS if args.case == "realistic" else c4["peak_steps"]
    t0 = time.perf_counter()
    res = o.trace(c4["a"], wl.R_OBS, c4["inc_deg"], c4["half_width"], 0, 0, seed=c4["seed"], idx=idx, h=wl.H,
                  cap_factor=wl.R_CAPTURE_FACTOR, esc_factor=wl.R_ESCAPE_FACTOR, rule=rule, max_steps=max_steps,
                  threads=threads, want_y0=False)
    dt = time.perf_counter() - t0
    return int(res["steps"].sum()), dt, m


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as o
    threads = max(1, o.hardware_threads())
    for _ in range(args.warmup):
        oracle_sample(args, args.ref_log2n, threads)
    tot_steps, tot_t = 0, 0.0
    for _ in range(args.steps):
        ps, dt, m = oracle_sample(args, args.ref_log2n, threads)
        tot_steps += ps
        tot_t += dt
    value = tot_steps / tot_t
    sample = f"{m} photons per step, strided p = j * 2^{args.log2n} / {m} from the same seeded workload"
    out = {"impl": "reference", "metric": "photon-steps/s", "value": value, "unit": "photon-steps/s", "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": workload_config(args, 1), "ns_per_photon_step": 1e9 / value,
           "cpu_baseline": {"value": value, "unit": "photon-steps/s", "cores": threads, "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": "photon-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def run_gray(args):
    import torch
    import torch.distributed as dist

    import paper_1303_5057_b200 as g
    from paper_1303_5057_b200 import workloads as wl

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libgray has no CPU path)")
    if args.share_gpu:
        local = 0
    torch.cuda.set_device(local)
    if world > 1:
        if args.dist_backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(args.dist_backend)
    dev = torch.device("cuda", local)

    c4 = wl.C4
    # 37 B (fp32) / 69 B (fp64) of state per photon, plus the e2e leg's device scratch: shrink the batch if it cannot fit
    per_photon = 38 if args.prec == "f32" else 70
    free_bytes, _ = torch.cuda.mem_get_info()
    if world > 1:
        fb = torch.tensor([free_bytes], dtype=torch.int64, device=dev)
        dist.all_reduce(fb, op=dist.ReduceOp.MIN)
        free_bytes = int(fb.item())
    while args.log2n > 20 and (2 ** args.log2n) * per_photon + (4 << 30) > free_bytes:
        args.log2n -= 1
    n = 2 ** args.log2n
    prec = g.GRAY_F32 if args.prec == "f32" else g.GRAY_F64
    rule = g.STEP_EQ2 if args.rule == "eq2" else g.STEP_REL
    peak_case = args.case == "peak"
    max_steps = c4["peak_steps"] if peak_case else wl.MAX_STEPS
    params = g.StepParams(h=wl.H, r_capture_factor=wl.R_CAPTURE_FACTOR, r_escape_factor=wl.R_ESCAPE_FACTOR, rule=rule,
                          schedule=g.SCHED_REFILL if args.schedule == "refill" else g.SCHED_STATIC,
                          refill_interval=args.refill_interval, frozen=peak_case,
                          photons_per_thread=args.photons_per_thread, xi_epsilon=args.xi_eps,
                          system=g.SYS_REDUCED if args.system == "reduced" else g.SYS_FULL)
    batch = g.PhotonBatch(n, prec, device=dev)
    p0 = rank * n                                   # weak scaling: every rank its own photon range

    kern_ev = []

    def step(timed):
        g.gray_init_rays_random(batch, c4["a"], wl.R_OBS, c4["inc_deg"], c4["half_width"], c4["seed"], p0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.gray_integrate(batch, max_steps=max_steps, params=params)
        e1.record()
        counts = g.gray_classify(batch)            # synchronises; the step's result on the host
        cnt = g.gray_integrate_counters(batch)
        if timed:
            kern_ev.append((e0, e1))
        return counts, cnt

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(False)
    sampler = ClockSampler(local) if rank == 0 else None
    barrier()
    t0 = time.perf_counter()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    photon_steps, issued, counts = 0, 0, None
    for _ in range(args.steps):
        counts, cnt = step(True)
        photon_steps += cnt["photon_steps"]
        issued += cnt["issued_steps"]
    ev1.record()
    barrier()
    t1 = time.perf_counter()
    clocks = sampler.stop(t0, t1) if sampler else None
    ms = ev0.elapsed_time(ev1)
    kern_ms = sum(a.elapsed_time(b) for a, b in kern_ev) / max(1, len(kern_ev))

    # ---- end to end through the C ABI with host buffers (copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        le = args.e2e_log2n if args.e2e_log2n >= 0 else min(args.log2n, 26)
        ne = 2 ** le
        dt = torch.float32 if prec == g.GRAY_F32 else torch.float64
        hb = g.PhotonBatch(ne, prec, device=dev)
        g.gray_init_rays_random(hb, c4["a"], wl.R_OBS, c4["inc_deg"], c4["half_width"], c4["seed"], p0)
        x_in, k_in = hb.x.cpu().pin_memory(), hb.k.cpu().pin_memory()
        del hb
        x_out, k_out = torch.empty_like(x_in).pin_memory(), torch.empty_like(k_in).pin_memory()
        st_h = torch.empty((ne,), dtype=torch.uint8).pin_memory()
        ns_h = torch.empty((ne,), dtype=torch.int32).pin_memory()
        chunk = min(ne, 1 << 23)
        scratch = torch.empty((g.gray_host_scratch_bytes(chunk, prec),), dtype=torch.uint8, device=dev)
        call = lambda: g.gray_integrate_host(x_in, k_in, x_out, k_out, st_h, ns_h, c4["a"], wl.R_OBS, max_steps=max_steps,
                                             params=params, chunk=chunk, scratch=scratch)
        call()                                                     # warm-up
        reps = max(1, min(args.steps, 3))
        barrier()
        w0 = time.perf_counter()
        e_steps = 0
        for _ in range(reps):
            e_steps += call()["photon_steps"]                      # synchronous: results are in host memory on return
        torch.cuda.synchronize()
        e_t = time.perf_counter() - w0
        h2d = int(x_in.numel() * x_in.element_size() * 2)
        d2h = int(h2d + st_h.numel() + ns_h.numel() * 4)
        e2e = {"steps_total": e_steps, "seconds": e_t, "h2d": h2d, "d2h": d2h, "photons": ne, "reps": reps}

    # ---- reduce over ranks: max time, summed work
    if world > 1:
        t = torch.tensor([ms, kern_ms, e2e["seconds"] if e2e else 0.0], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms, kern_ms = float(t[0]), float(t[1])
        s = torch.tensor([photon_steps, issued, e2e["steps_total"] if e2e else 0], dtype=torch.float64, device=dev)
        dist.all_reduce(s, op=dist.ReduceOp.SUM)
        if e2e:
            e2e["seconds"] = float(t[2])
            e2e["steps_total"] = float(s[2])
        tot_steps, tot_issued = float(s[0]), float(s[1])
    else:
        tot_steps, tot_issued = float(photon_steps), float(issued)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = tot_steps / (ms * 1e-3)
    flops = FLOPS_PER_PHOTON_STEP[args.rule]
    # roofline of the dominant kernel (integrate_kernel), per GPU: algorithmic flops per launch / its duration
    per_gpu_steps = tot_steps / world / args.steps
    counted = per_gpu_steps if not peak_case else tot_issued / world / args.steps   # peak case: every issued lane-step computes
    achieved = flops * counted / (kern_ms * 1e-3) / 1e12
    peak = PEAK_TFLOPS[args.prec]
    fma_peak = g.gray_fma_peak(prec, 8192) / 1e12
    # Achievable ceiling of the packed fp32 kernel: the FP32 pipe retires the
    # integrator's mix of FMUL2 / FFMA2 / FADD2 with changing register operands at this fraction of its lane rate
    mix = None
    if args.prec == "f32" and args.photons_per_thread != 1:
        lane_peak = 148 * 128 * 1.965e9
        mix = {"ffma2_invariant_operands": g.gray_packed_peak(0) / lane_peak, "ffma2_three_register_pairs": g.gray_packed_peak(1) / lane_peak,
               "integrator_mix": g.gray_packed_peak(2) / lane_peak}
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": (NCU_DRAM_BYTES_PER_PHOTON * n) if (NCU_DRAM_BYTES_PER_PHOTON and args.prec == "f32") else None,
                "traffic_source": "ncu dram bytes per photon of the 2^30-photon launch (profiles/) x photons of this launch",
                "kernel": "gray::integrate_kernel", "kernel_ms": kern_ms, "kernel_share_of_step": kern_ms * args.steps / ms,
                "executed_flops_per_photon_step": NCU_EXECUTED_FLOPS_PER_PHOTON_STEP if (args.prec == "f32" and args.photons_per_thread != 1 and args.system == "full" and args.xi_eps == 0) else None,
                "flops_per_photon_step": flops, "flops_source": "oracle operation tally (add=sub=mul=div=sqrt=sin=cos=1)",
                "peak_source": "148 SMs x %d lanes x 2 x 1.965 GHz (DESIGN.md)" % (128 if args.prec == "f32" else 64),
                "fma_microbench_tflops": fma_peak, "frac_of_fma_microbench": achieved / fma_peak,
                "lane_efficiency": tot_steps / tot_issued if tot_issued else None,
                "packed_pipe_fraction_measured": mix,
                "frac_of_achievable": (achieved / peak) / (mix["integrator_mix"] * 787.0 / 792.0) if mix else None,
                "hbm_algorithmic_bytes_per_launch": n * (2 * (32 if args.prec == "f32" else 64) + 10)}
    if args.system == "reduced":
        # the operation tally is the full system's; the reduced system does less work per step, so a FLOP rate
        # against that tally would overstate it: only photon-steps/s is reported for it
        for k in ("achieved", "frac", "frac_of_fma_microbench", "frac_of_achievable"):
            roofline[k] = None
        roofline["note"] = "system=reduced: no operation tally of its own; see value / ns_per_photon_step"
    out = {"metric": "photon-steps/s", "value": value, "unit": "photon-steps/s", "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": args.prec, "data": "synthetic", "config": workload_config(args, world),
           "ns_per_photon_step": 1e9 / value, "gflops": flops * value / 1e9 if args.system == "full" else None,
           "mean_steps_per_photon": tot_steps / (world * n * args.steps), "status_counts_rank0": counts,
           "roofline": roofline, "gpu_launches": 3 * args.steps, "clocks": clocks,
           "paper_context": "GRay on Tesla M2090 (2013): 1.15 ns/photon/step single precision, >300 GFLOP/s (P:7, P:150)"}
    if e2e:
        out["e2e"] = {"value": e2e["steps_total"] / e2e["seconds"], "unit": "photon-steps/s",
                      "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"],
                      "photons_per_gpu": e2e["photons"], "reps": e2e["reps"],
                      "call": "gray_integrate_host (pinned host x,k in; x,k,status,steps out; 2^23-photon chunks on two streams)",
                      "timer": "host wall clock around the synchronous C-ABI calls"}
    if not args.no_cpu_baseline:
        import oracle as o                          # cpu_baseline leg only
        threads = max(1, o.hardware_threads())
        ps, dt, m = oracle_sample(args, 18, threads)
        out["cpu_baseline"] = {"value": ps / dt, "unit": "photon-steps/s", "cores": threads, "kind": "oracle",
                               "sample": f"{m} photons, strided p = j * 2^{args.log2n} / {m} of rank 0's photons, "
                                         f"{ps} photon-steps in {dt:.1f} s", "ns_per_photon_step_per_core": 1e9 * dt * threads / ps}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_projection(args):
    """Paper's Fig. 4: run time of the equatorial-plane grid projection, a = 0.95, i = 60 deg, against
    the number of rays n (square grids over +-10 M).  Host wall clock around init -> integrate -> counters (what a
    user waits for), best of 5; the paper finds a launch floor of ~20 ms and linear growth beyond ~1e4 rays on its
    Tesla M2090 in double precision."""
    import torch

    import paper_1303_5057_b200 as g
    from paper_1303_5057_b200 import workloads as wl
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    if int(os.environ.get("RANK", "0")) != 0:
        return
    rows = []
    for prec_name, prec in (("f64", g.GRAY_F64), ("f32", g.GRAY_F32)):
        for log2n in range(8, 27, 2):
            side = 2 ** (log2n // 2)
            b = g.PhotonBatch(side * side, prec)
            params = g.StepParams(rule=g.STEP_EQ2, stop_at_equator=True)
            best, steps = 1e30, 0
            for rep in range(6):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                g.gray_init_rays(b, 0.95, wl.R_OBS, 60.0, 10.0, side, side)
                g.gray_integrate(b, max_steps=wl.MAX_STEPS, params=params)
                steps = g.gray_integrate_counters(b)["photon_steps"]          # synchronises
                dt = time.perf_counter() - t0
                if rep:
                    best = min(best, dt)
            rows.append({"precision": prec_name, "rays": side * side, "ms": 1e3 * best, "photon_steps": steps,
                         "ns_per_photon_step": 1e9 * best / max(1, steps)})
    out = {"metric": "run time of the equatorial-plane grid projection vs number of rays", "unit": "ms", "n_gpus": 1,
           "data": "synthetic", "higher_is_better": False,
           "config": {"workload": "paper Fig. 4: a=0.95, i=60 deg, square grids over +-10 M at r_obs=1000 M, eq. (2) rule, "
                                  "stop at the equatorial plane", "timer": "host wall clock, best of 5"},
           "rows": rows, "paper_context": "Tesla M2090, double precision: ~20 ms floor below ~1e4 rays, then linear (P:136-138)"}
    print(json.dumps(out), flush=True)


def main():
    args = parse()
    if args.case == "projection" and args.impl != "reference":
        run_projection(args)
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gray(args)


if __name__ == "__main__":
    main()
