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
# The same tally of the oracle's reduced system (oracle.op_tally(..., system=SYS_REDUCED)).  Its formulation rebuilds
# k^t, k^phi from E, L in every stage and then evaluates the FULL right-hand side, two equations of which it throws away
# (gray_oracle.hpp rhs_reduced): 920 > 787, although the reduced kernel executes about 0.8 of the full one's instructions.
# A fraction by this tally can exceed 1; it is printed because BASELINE defines the fraction by the oracle's tally, and
# `frac_executed` beside it is the hardware-side figure.
FLOPS_PER_PHOTON_STEP_REDUCED = {"rel": 910, "eq2": 920}
# FP32 CUDA-core peak the integrator is bound by: 148 SMs x 128 lanes x 2 (FMA) x
# 1.965 GHz (clocks.max.sm); FP64: 64 lanes per SM.
PEAK_TFLOPS = {"f32": 148 * 128 * 2 * 1.965e9 / 1e12, "f64": 148 * 64 * 2 * 1.965e9 / 1e12}
# The survey's own hand count of a photon-step in the collected-term formulation (655 + 8 trig),
# a third reading next to the oracle's tally and the executed count
FLOPS_SURVEY_HAND_TALLY = 663


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
    ap.add_argument("--case", default="realistic", choices=["realistic", "peak", "projection", "ring", "survey"],
                    help="projection = the paper's first benchmark (P:130-140, Fig. 4): run time of the grid projection "
                         "onto the equatorial plane (a = 0.95, i = 60 deg) against the number of rays; ring = the paper's "
                         "photon-ring study (section 4, P:165-210): 16 spins x 19 inclinations x 6000 x 181 rays; survey = "
                         "BASELINE config C5: 11 spins x 9 inclinations, 1024 x 1024 images, shadow statistics per case")
    ap.add_argument("--schedule", default="refill", choices=["refill", "static"])
    ap.add_argument("--refill-interval", type=int, default=0)
    ap.add_argument("--photons-per-thread", type=int, default=0, help="0 = library default (2 for f32: packed FFMA2), 1, 2")
    ap.add_argument("--system", default="full", choices=["full", "reduced"], help="full = the 8 second-order equations of the north star; reduced = E, L_z eliminate k^t, k^phi")
    ap.add_argument("--xi-eps", type=float, default=0.0, help="epsilon of the paper's xi monitor (P:107); 0 = off")
    ap.add_argument("--e2e-log2n", type=int, default=-1, help="photons per GPU of the host-buffer run (default min(log2n, 28), lowered if the host "
                    "cannot pin the buffers)")
    ap.add_argument("--no-secondary", action="store_true", help="skip the secondary measurements (C4 sweep, peak case, fp64, xi, reduced)")
    ap.add_argument("--cpu-log2n", type=int, default=21, help="photons of the oracle's all-core sample (the one-core sample has 1/16 of it)")
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
    # (rule first, under 120 characters: the driver's record keeps that much of the string)
    return {"workload": f"C4-{args.case} rule={args.rule}: 2^{args.log2n} photons/GPU, Kerr a={c4['a']} i={c4['inc_deg']:g} deg, "
                        f"random pixels +-{c4['half_width']:g} M, r_obs={wl.R_OBS:.0f} M, RK4 h=1/32",
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
           "config": workload_config(args, 1),
           "note": "the oracle computes in f64 (dtype) whatever config.precision says: that key names the GPU arm's build",
           "ns_per_photon_step": 1e9 / value,
           "cpu_baseline": {"value": value, "unit": "photon-steps/s", "cores": threads, "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": "photon-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def read_profile_csv(name):
    """Rows of a committed ncu CSV under profiles/ (lines before the header are ncu's own banner)."""
    import csv
    path = os.path.join(ROOT, "profiles", name)
    if not os.path.exists(path):
        return None
    with open(path) as f:
        lines = [l for l in f if l.startswith('"')]
    return list(csv.DictReader(lines))


def ncu_dram_bytes_per_photon():
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE gray_integrate launch of the default workload (2^30 photons,
    fp32), read from the committed ncu capture: (bytes per photon, file name).  Not a measurement of this run."""
    for name in ("r02_integrate_f2_dram_2p30.csv", "r01_integrate_f2_dram_2p30.csv"):
        rows = read_profile_csv(name)
        if not rows:
            continue
        tot = sum(float(r["Metric Value"].replace(",", "")) for r in rows if r["Metric Name"].startswith("dram__bytes_"))
        if tot > 0:
            return tot / 2 ** 30, name
    return None, None


def executed_flops_per_lane_step(variant):
    """FP operations the kernel variant EXECUTES per issued lane-step (one RK4 step of one photon slot, whether or not
    the slot holds a live photon; FMA = 2), from the per-opcode executed thread-instruction counts of the committed ncu
    captures (profiles/r02_executed_ops.csv); None if the variant was not captured."""
    rows = read_profile_csv("r02_executed_ops.csv")
    for r in rows or []:
        if r["variant"] == variant:
            return float(r["flops_per_issued_lane_step"])
    return None


def variant_name(prec, rule, case, xi_eps, system, ppt):
    v = "f64" if prec == "f64" else ("f32x1" if ppt == 1 else "f32")
    v += "_" + rule
    if case == "peak":
        v += "_frozen"
    if xi_eps > 0:
        v += "_xi"
    if system == "reduced":
        v += "_reduced"
    return v


class Runner:
    """Times bench steps (init -> integrate -> classify) of one workload variant on this rank's GPU."""

    def __init__(self, args):
        import torch
        import torch.distributed as dist

        import paper_1303_5057_b200 as g
        from paper_1303_5057_b200 import workloads as wl
        self.torch, self.dist, self.g, self.wl = torch, dist, g, wl
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py: no CUDA device (libgray has no CPU path)")
        if args.share_gpu:
            local = 0
        self.local = local
        torch.cuda.set_device(local)
        if self.world > 1:
            if args.dist_backend == "nccl":
                dist.init_process_group("nccl", device_id=torch.device("cuda", local))
            else:
                dist.init_process_group(args.dist_backend)
        self.dev = torch.device("cuda", local)

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def fit_log2n(self, log2n, prec):
        """37 B (fp32) / 69 B (fp64) of state per photon plus head room: shrink the batch if the device cannot hold it."""
        per_photon = 38 if prec == "f32" else 70
        free_bytes, _ = self.torch.cuda.mem_get_info()
        if self.world > 1:
            fb = self.torch.tensor([free_bytes], dtype=self.torch.int64, device=self.dev)
            self.dist.all_reduce(fb, op=self.dist.ReduceOp.MIN)
            free_bytes = int(fb.item())
        while log2n > 20 and (2 ** log2n) * per_photon + (4 << 30) > free_bytes:
            log2n -= 1
        return log2n

    def params(self, rule, case, xi_eps, system, ppt, schedule="refill", refill_interval=0):
        g, wl = self.g, self.wl
        return g.StepParams(h=wl.H, r_capture_factor=wl.R_CAPTURE_FACTOR, r_escape_factor=wl.R_ESCAPE_FACTOR,
                            rule=g.STEP_EQ2 if rule == "eq2" else g.STEP_REL,
                            schedule=g.SCHED_REFILL if schedule == "refill" else g.SCHED_STATIC,
                            refill_interval=refill_interval, frozen=(case == "peak"), photons_per_thread=ppt,
                            xi_epsilon=xi_eps, system=g.SYS_REDUCED if system == "reduced" else g.SYS_FULL)

    def run(self, *, log2n, prec, rule, case, xi_eps=0.0, system="full", ppt=0, schedule="refill", refill_interval=0,
            steps, warmup, sample_clocks=False):
        """W untimed + K timed bench steps; returns the per-rank-reduced measurement (max time, summed work)."""
        torch, g, wl = self.torch, self.g, self.wl
        c4 = wl.C4
        n = 2 ** log2n
        gprec = g.GRAY_F32 if prec == "f32" else g.GRAY_F64
        max_steps = c4["peak_steps"] if case == "peak" else wl.MAX_STEPS
        params = self.params(rule, case, xi_eps, system, ppt, schedule, refill_interval)
        batch = g.PhotonBatch(n, gprec, device=self.dev)
        p0 = self.rank * n                                   # weak scaling: every rank its own photon range
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

        for _ in range(warmup):
            step(False)
        sampler = ClockSampler(self.local) if (sample_clocks and self.rank == 0) else None
        self.barrier()
        t0 = time.perf_counter()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        photon_steps, issued, counts = 0, 0, None
        for _ in range(steps):
            counts, cnt = step(True)
            photon_steps += cnt["photon_steps"]
            issued += cnt["issued_steps"]
        ev1.record()
        self.barrier()
        t1 = time.perf_counter()
        clocks = sampler.stop(t0, t1) if sampler else None
        ms = ev0.elapsed_time(ev1)
        kern_ms = sum(a.elapsed_time(b) for a, b in kern_ev) / max(1, len(kern_ev))
        del batch
        if self.world > 1:
            t = torch.tensor([ms, kern_ms], dtype=torch.float64, device=self.dev)
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
            ms, kern_ms = float(t[0]), float(t[1])
            w = torch.tensor([photon_steps, issued], dtype=torch.float64, device=self.dev)
            self.dist.all_reduce(w, op=self.dist.ReduceOp.SUM)
            photon_steps, issued = float(w[0]), float(w[1])
        return dict(n=n, log2n=log2n, prec=prec, rule=rule, case=case, xi_eps=xi_eps, system=system, ppt=ppt, steps=steps,
                    ms=ms, kernel_ms=kern_ms, photon_steps=float(photon_steps), issued=float(issued), counts=counts,
                    clocks=clocks, max_steps=max_steps)

    def roofline(self, m):
        """Roofline fields of the dominant kernel (integrate_kernel) of a measurement, per GPU: work per launch / its
        CUDA-event duration against the FMA peak.  `frac` counts the oracle's operation tally (BASELINE's definition),
        `frac_executed` the operations the kernel executes (ncu), both with FMA = 2."""
        per_gpu_steps = m["photon_steps"] / self.world / m["steps"]
        # peak case: every issued lane-step computes, so issued lane-steps are the units
        counted = per_gpu_steps if m["case"] != "peak" else m["issued"] / self.world / m["steps"]
        peak = PEAK_TFLOPS[m["prec"]]
        rate = counted / (m["kernel_ms"] * 1e-3)                        # units per second inside the kernel
        reduced = m["system"] == "reduced"
        flops = (FLOPS_PER_PHOTON_STEP_REDUCED if reduced else FLOPS_PER_PHOTON_STEP)[m["rule"]]
        achieved = flops * rate / 1e12
        exe = executed_flops_per_lane_step(variant_name(m["prec"], m["rule"], m["case"], m["xi_eps"], m["system"], m["ppt"]))
        issued_rate = m["issued"] / self.world / m["steps"] / (m["kernel_ms"] * 1e-3)       # lane-steps per second inside the kernel
        return dict(achieved=achieved, peak=peak, frac=achieved / peak, flops_per_photon_step=flops,
                    executed_flops_per_lane_step=exe, achieved_executed=exe * issued_rate / 1e12 if exe else None,
                    frac_executed=exe * issued_rate / 1e12 / peak if exe else None,
                    frac_survey_hand_tally=None if (reduced or m["prec"] != "f32") else FLOPS_SURVEY_HAND_TALLY * rate / 1e12 / peak,
                    kernel_ms=m["kernel_ms"], kernel_share_of_step=m["kernel_ms"] * m["steps"] / m["ms"],
                    lane_efficiency=m["photon_steps"] / m["issued"] if m["issued"] else None)


def secondary_line(R, m, label):
    rf = R.roofline(m)
    value = m["photon_steps"] / (m["ms"] * 1e-3)
    return {"workload": label, "dtype": m["prec"], "photons_per_gpu": m["n"], "steps": m["steps"], "value": value,
            "unit": "photon-steps/s", "ns_per_photon_step": 1e9 / value, "kernel_ms": rf["kernel_ms"],
            "frac": rf["frac"], "flops_per_photon_step": rf["flops_per_photon_step"], "frac_executed": rf["frac_executed"],
            "lane_efficiency": rf["lane_efficiency"],
            "issued_lane_steps_per_s": m["issued"] / (m["ms"] * 1e-3)}


def run_e2e(R, args, params, max_steps, prec, p0):
    """The same metric end to end through the C ABI with HOST buffers (gray_integrate_host): pinned host x, k in;
    x, k, status, steps out; both copies inside the timed region."""
    torch, g, wl = R.torch, R.g, R.wl
    c4 = wl.C4
    gprec = g.GRAY_F32 if prec == "f32" else g.GRAY_F64
    bytes_per_photon = (2 * 32 if prec == "f32" else 2 * 64) * 2 + 5        # pinned: inputs, outputs, status, steps
    le = args.e2e_log2n if args.e2e_log2n >= 0 else min(args.log2n, 28)
    note = None
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:  # pragma: no cover
        avail = 16 << 30
    while le > 20 and 1.25 * bytes_per_photon * 2 ** le * (R.world if args.share_gpu or R.world > 1 else 1) > avail:
        le -= 1
        note = "reduced to fit the host's available memory (%.0f GB) with pinned in + out buffers" % (avail / 2 ** 30)
    ne = 2 ** le
    dt = torch.float32 if prec == "f32" else torch.float64
    x_in = torch.empty((ne, 4), dtype=dt, pin_memory=True)
    k_in = torch.empty((ne, 4), dtype=dt, pin_memory=True)
    piece = min(ne, 1 << 26)
    hb = g.PhotonBatch(piece, gprec, device=R.dev)
    for lo in range(0, ne, piece):                                  # initial states, made on the device piecewise
        g.gray_init_rays_random(hb, c4["a"], wl.R_OBS, c4["inc_deg"], c4["half_width"], c4["seed"], p0 + lo)
        x_in[lo:lo + piece].copy_(hb.x)
        k_in[lo:lo + piece].copy_(hb.k)
    del hb
    x_out, k_out = torch.empty_like(x_in, pin_memory=True), torch.empty_like(k_in, pin_memory=True)
    st_h = torch.empty((ne,), dtype=torch.uint8, pin_memory=True)
    ns_h = torch.empty((ne,), dtype=torch.int32, pin_memory=True)
    chunk = min(ne, 1 << 23)
    scratch = torch.empty((g.gray_host_scratch_bytes(chunk, gprec),), dtype=torch.uint8, device=R.dev)
    call = lambda: g.gray_integrate_host(x_in, k_in, x_out, k_out, st_h, ns_h, c4["a"], wl.R_OBS, max_steps=max_steps,
                                         params=params, chunk=chunk, scratch=scratch)
    call()                                                     # warm-up (also creates the library's two streams)
    reps = max(1, min(args.steps, 2 if le >= 28 else 3))
    R.barrier()
    w0 = time.perf_counter()
    e_steps = 0
    for _ in range(reps):
        e_steps += call()["photon_steps"]                      # synchronous: results are in host memory on return
    torch.cuda.synchronize()
    e_t = time.perf_counter() - w0
    h2d = int(x_in.numel() * x_in.element_size() * 2)
    d2h = int(h2d + st_h.numel() + ns_h.numel() * 4)
    if R.world > 1:
        t = torch.tensor([e_t], dtype=torch.float64, device=R.dev)
        R.dist.all_reduce(t, op=R.dist.ReduceOp.MAX)
        w = torch.tensor([e_steps], dtype=torch.float64, device=R.dev)
        R.dist.all_reduce(w, op=R.dist.ReduceOp.SUM)
        e_t, e_steps = float(t[0]), float(w[0])
    return {"value": e_steps / e_t, "unit": "photon-steps/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
            "photons_per_gpu": ne, "reps": reps, "note": note,
            "call": "gray_integrate_host (pinned host x,k in; x,k,status,steps out; 2^23-photon chunks on two streams)",
            "timer": "host wall clock around the synchronous C-ABI calls"}


def run_gray(args):
    R = Runner(args)
    g, wl = R.g, R.wl
    world, rank = R.world, R.rank
    args.log2n = R.fit_log2n(args.log2n, args.prec)
    n = 2 ** args.log2n
    prec = g.GRAY_F32 if args.prec == "f32" else g.GRAY_F64

    # ---- the headline: BASELINE's metric on config C4 at its largest size
    m = R.run(log2n=args.log2n, prec=args.prec, rule=args.rule, case=args.case, xi_eps=args.xi_eps, system=args.system,
              ppt=args.photons_per_thread, schedule=args.schedule, refill_interval=args.refill_interval, steps=args.steps,
              warmup=args.warmup, sample_clocks=True)

    # ---- end to end through the C ABI with host buffers (copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        params = R.params(args.rule, args.case, args.xi_eps, args.system, args.photons_per_thread, args.schedule, args.refill_interval)
        e2e = run_e2e(R, args, params, m["max_steps"], args.prec, rank * n)

    # ---- every other quoted number, in the same run: C4's sweep in both cases, fp64, xi monitor,
    #      reduced system; 1 warm-up + 2 timed steps each
    secondary = []
    if not args.no_secondary:
        todo = []
        for l2 in (20, 24, 28):
            if l2 < args.log2n or args.case != "realistic":
                todo.append((f"C4-realistic 2^{l2} photons/GPU, fp32, eq2", dict(log2n=l2, prec="f32", rule="eq2", case="realistic")))
        for l2 in (20, 24, 28):
            todo.append((f"C4-peak 2^{l2} photons/GPU: {wl.C4['peak_steps']} REL steps per lane, state frozen by select (R17)",
                         dict(log2n=l2, prec="f32", rule="rel", case="peak")))
        todo.append(("C4-realistic 2^26 photons/GPU, fp64 build, eq2", dict(log2n=26, prec="f64", rule="eq2", case="realistic")))
        todo.append(("C4-realistic 2^26 photons/GPU, fp32, eq2, xi monitor eps=1e-3 (paper's production scheme, P:103-109)",
                     dict(log2n=26, prec="f32", rule="eq2", case="realistic", xi_eps=1e-3)))
        todo.append(("C4-realistic 2^26 photons/GPU, fp32, eq2, reduced system (E, L_z eliminate k^t, k^phi)",
                     dict(log2n=26, prec="f32", rule="eq2", case="realistic", system="reduced")))
        todo.append(("C4-realistic 2^26 photons/GPU, fp32, eq2, one photon per thread (scalar FFMA)",
                     dict(log2n=26, prec="f32", rule="eq2", case="realistic", ppt=1)))
        for label, kw in todo:
            kw["log2n"] = min(kw["log2n"], R.fit_log2n(kw["log2n"], kw["prec"]))
            ms = R.run(steps=2, warmup=1, **kw)
            if rank == 0:
                secondary.append(secondary_line(R, ms, label))

    if rank != 0:
        if world > 1:
            R.dist.destroy_process_group()
        return

    value = m["photon_steps"] / (m["ms"] * 1e-3)
    rf = R.roofline(m)
    fma_peak = g.gray_fma_peak(prec, 8192) / 1e12
    mix = None
    if args.prec == "f32" and args.photons_per_thread != 1:
        lane_peak = 148 * 128 * 1.965e9
        mix = {"ffma2_invariant_operands": g.gray_packed_peak(0) / lane_peak, "ffma2_three_register_pairs": g.gray_packed_peak(1) / lane_peak,
               "ffma2_two_register_pairs": g.gray_packed_peak(4) / lane_peak, "fmul2_two_register_pairs": g.gray_packed_peak(3) / lane_peak,
               "integrator_mix_r01": g.gray_packed_peak(2) / lane_peak, "integrator_packed_mix": g.gray_packed_peak(5) / lane_peak,
               "integrator_packed_mix_with_its_other_instructions": g.gray_packed_peak(6) / lane_peak}
    dram_b, dram_src = ncu_dram_bytes_per_photon()
    flops = FLOPS_PER_PHOTON_STEP[args.rule]
    roofline = {"bound": "alu", "achieved": rf["achieved"], "peak": rf["peak"], "unit": "TFLOP/s", "frac": rf["frac"],
                "traffic": (dram_b * n) if (dram_b and args.prec == "f32") else None,
                "traffic_source": (f"NOT measured in this run: ncu dram bytes per photon of one 2^30-photon launch, read from profiles/{dram_src}, "
                                   "x photons of this launch") if dram_b else None,
                "kernel": "gray::integrate_kernel", "kernel_ms": rf["kernel_ms"], "kernel_share_of_step": rf["kernel_share_of_step"],
                "flops_per_photon_step": flops, "flops_source": "oracle operation tally (add=sub=mul=div=sqrt=sin=cos=1): BASELINE's definition",
                "executed_flops_per_lane_step": rf["executed_flops_per_lane_step"],
                "executed_source": "ncu per-opcode executed thread-instruction counts per issued lane-step (profiles/r02_executed_ops.csv), "
                                   "FMA = 2, x issued lane-steps of this run",
                "achieved_executed": rf["achieved_executed"], "frac_executed": rf["frac_executed"],
                "flops_survey_hand_tally": FLOPS_SURVEY_HAND_TALLY, "frac_survey_hand_tally": rf["frac_survey_hand_tally"],
                "peak_source": "148 SMs x %d lanes x 2 x 1.965 GHz (DESIGN.md)" % (128 if args.prec == "f32" else 64),
                "fma_microbench_tflops": fma_peak, "frac_of_fma_microbench": rf["achieved"] / fma_peak if rf["achieved"] else None,
                "lane_efficiency": rf["lane_efficiency"], "packed_pipe_fraction_measured": mix,
                "hbm_algorithmic_bytes_per_launch": n * (2 * (32 if args.prec == "f32" else 64) + 10)}
    if args.system == "reduced":
        roofline["flops_per_photon_step"] = rf["flops_per_photon_step"]
        roofline["note"] = ("system=reduced: the oracle's reduced formulation tallies more operations per step than its full one "
                            "(it evaluates the full right-hand side and discards two equations), so frac can exceed 1; see frac_executed")
    out = {"metric": "photon-steps/s", "value": value, "unit": "photon-steps/s", "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": m["ms"] / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": args.prec, "data": "synthetic", "config": workload_config(args, world),
           "ns_per_photon_step": 1e9 / value, "gflops": flops * value / 1e9 if args.system == "full" else None,
           "mean_steps_per_photon": m["photon_steps"] / (world * n * args.steps), "status_counts_rank0": m["counts"],
           "roofline": roofline, "gpu_launches": 3 * args.steps, "clocks": m["clocks"],
           "paper_context": "GRay on Tesla M2090 (2013): 1.15 ns/photon/step single precision, >300 GFLOP/s (P:7, P:150)"}
    if e2e:
        out["e2e"] = e2e
    if secondary:
        out["secondary"] = secondary
    if not args.no_secondary and world == 1:
        # the applications this repository quotes, in the same run: BASELINE config C5 and the paper's photon-ring study
        apps = []
        for fn in (run_survey, run_ring):
            a = fn(args, emit=False)
            apps.append({k: a[k] for k in ("metric", "value", "unit", "geodesics", "geodesics_per_s", "photon_steps", "photon_steps_per_s", "config")})
        out["applications"] = apps
    if not args.no_cpu_baseline:
        import oracle as o                          # cpu_baseline leg only
        threads = max(1, o.hardware_threads())
        ps, dt, mm = oracle_sample(args, args.cpu_log2n, threads)
        ps1, dt1, m1 = oracle_sample(args, max(10, args.cpu_log2n - 4), 1)
        out["cpu_baseline"] = {"value": ps / dt, "unit": "photon-steps/s", "cores": threads, "kind": "oracle",
                               "sample": f"{mm} photons, strided p = j * 2^{args.log2n} / {mm} of rank 0's photons, "
                                         f"{ps} photon-steps in {dt:.1f} s",
                               "ns_per_photon_step": 1e9 * dt / ps,
                               "one_core": {"value": ps1 / dt1, "unit": "photon-steps/s", "cores": 1, "ns_per_photon_step": 1e9 * dt1 / ps1,
                                            "sample": f"{m1} photons of the same strided sample, {ps1} photon-steps in {dt1:.1f} s"}}
        # like for like next to the mixed-precision ratio: the oracle computes in fp64, so the fp64 build is its
        # counterpart; vs_baseline stays null (BASELINE.md holds no published number for this metric and workload)
        f64 = [s2["value"] for s2 in secondary if s2["dtype"] == "f64"] if secondary else []
        out["cpu_baseline"]["gpu_over_oracle"] = {"this_line_%s" % args.prec: value / (ps / dt),
                                                  "f64_build_same_run": (f64[0] / (ps / dt)) if f64 else None}
    print(json.dumps(out), flush=True)
    if world > 1:
        R.dist.destroy_process_group()


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


def run_ring(args, emit=True):
    """Paper section 4: the photon ring of a Kerr black hole for 16 spins a_j = 1 - 10^(-j/5) and 19
    inclinations 0, 5, ..., 90 deg, each image a polar grid of 6000 x 181 rays over (1.5 M, 7.5 M) x [0, pi] at
    r_obs = 1000 M (3.3e8 geodesics), with the xi monitor on as in the paper: init -> integrate -> ring statistics
    (D, <R>, A of eqs. 6-8) per case.  Timed with CUDA events over the whole study; tests/test_gpu_configs.py compares every
    case with the closed-form Bardeen curve and the oracle."""
    import torch

    import paper_1303_5057_b200 as g
    from paper_1303_5057_b200 import workloads as wl
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    if int(os.environ.get("RANK", "0")) != 0:
        return
    R_lo, R_hi, n_R, n_th = 1.5, 7.5, 6000, 181
    n_img = n_R * n_th
    incs = list(range(0, 91, 5))
    # the 19 images of one spin differ only in the inclination, which the integrator does not read: they are initialised
    # slice by slice, integrated in ONE launch (2.06e7 rays keep the persistent grid full) and evaluated slice by slice
    big = g.PhotonBatch(n_img * len(incs), g.GRAY_F32)
    views = [big.slice(i * n_img, (i + 1) * n_img) for i in range(len(incs))]
    params = g.StepParams(rule=g.STEP_EQ2, xi_epsilon=1e-3)
    show = {(0, 0), (0, 60), (5, 60), (10, 30), (10, 60), (10, 90), (15, 0), (15, 60), (15, 90)}
    rows, steps, fallback, lost = [], 0, 0, 0

    def study(record):
        nonlocal steps, fallback, lost
        for j in range(16):
            a = 1.0 - 10.0 ** (-j / 5.0)
            for v, inc in zip(views, incs):
                g.gray_init_rays_polar(v, a, wl.R_OBS, float(inc), R_lo, R_hi, n_R, n_th)
            big.set_image_plane(a, wl.R_OBS, 0.0, R_hi)
            g.gray_integrate(big, max_steps=wl.MAX_STEPS, params=params)
            if record:
                c = g.gray_integrate_counters(big)
                steps += c["photon_steps"]
                fallback += c["fallback_steps"]
            for v, inc in zip(views, incs):
                s = g.gray_ring_polar(v, None, bridge_axis=True)           # synchronises: the image's result on the host
                if record:
                    lost += s["axis_rays_lost"]
                    if (j, inc) in show:
                        rows.append({"a": round(a, 6), "inc_deg": inc, "D": s["D"], "R_mean": s["R_mean"], "A": s["A"],
                                     "alpha_min": s["alpha_min"], "alpha_max": s["alpha_max"]})

    study(False)                                                           # warm-up pass
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    study(True)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    n_geo = 16 * 19 * n_R * n_th
    out = {"metric": "run time of the paper's photon-ring study (section 4)", "unit": "s", "value": ms * 1e-3, "n_gpus": 1,
           "higher_is_better": False, "data": "synthetic", "dtype": "f32",
           "config": {"workload": "304 images (16 spins a_j = 1 - 10^(-j/5) x 19 inclinations 0..90 deg), polar grid 6000 x 181 rays over "
                                  "(1.5, 7.5) M x [0, pi] at r_obs = 1000 M, eq. (2) rule h = 1/32, xi monitor eps = 1e-3",
                      "timer": "CUDA events around the whole study (per spin: 19 x init, one integrate launch over the 19 images, 19 x ring statistics read back), after one warm-up pass"},
           "geodesics": n_geo, "geodesics_per_s": n_geo / (ms * 1e-3), "photon_steps": steps, "photon_steps_per_s": steps / (ms * 1e-3),
           "xi_fallback_steps": fallback, "axis_rays_lost": lost, "rows": rows,
           "paper_context": "16 x 19 x 6000 x 181 ~ 3e8 geodesics, 'none of them fails at the pole' (P:109, P:170); ring radius ~ 5.2 M, "
                            "nearly circular up to a ~ 0.9 (P:172-174)"}
    del big, views
    if emit:
        print(json.dumps(out), flush=True)
    return out


def run_survey(args, emit=True):
    """BASELINE config C5: the shadow / photon-ring survey, spins {0, 0.1, ..., 0.9, 0.99} x inclinations {5, 15, ..., 85} deg
    (99 cases), each a 1024 x 1024 image over +-10 M at r_obs = 1000 M, fp32, eq. (2) rule, xi monitor on; per case the
    capture map, shadow area, centroid, D, <R>, A and the boundary radius on 360 spokes (gray_classify + gray_shadow_edge).
    The nine images of a spin share one integrate launch (PhotonBatch.slice)."""
    import torch

    import paper_1303_5057_b200 as g
    from paper_1303_5057_b200 import workloads as wl
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    if int(os.environ.get("RANK", "0")) != 0:
        return
    c5 = wl.C5
    nx, ny, W = c5["nx"], c5["ny"], c5["half_width"]
    n_img = nx * ny
    incs = c5["incs_deg"]
    big = g.PhotonBatch(n_img * len(incs), g.GRAY_F32)
    views = [big.slice(i * n_img, (i + 1) * n_img) for i in range(len(incs))]
    cmap = torch.empty((ny, nx), dtype=torch.uint8, device="cuda")
    radius = torch.empty((360,), dtype=torch.float64, device="cuda")
    params = g.StepParams(rule=g.STEP_EQ2, xi_epsilon=1e-3)
    show = {(0.0, 45.0), (0.5, 45.0), (0.9, 5.0), (0.9, 45.0), (0.9, 85.0), (0.99, 45.0), (0.99, 85.0)}
    rows, steps, bad = [], 0, 0

    def study(record):
        nonlocal steps, bad
        for a in c5["spins"]:
            for v, inc in zip(views, incs):
                g.gray_init_rays(v, a, wl.R_OBS, inc, W, nx, ny)
            big.set_image_plane(a, wl.R_OBS, 0.0, W)
            g.gray_integrate(big, max_steps=wl.MAX_STEPS, params=params)
            if record:
                steps += g.gray_integrate_counters(big)["photon_steps"]
            for v, inc in zip(views, incs):
                counts = g.gray_classify(v, cmap)
                s = g.gray_shadow_edge(v, 360, radius)                     # synchronises: the image's result on the host
                if record:
                    bad += counts[g.BAD] + counts[g.LIVE]
                    if (a, inc) in show:
                        rows.append({"a": a, "inc_deg": inc, "captured": counts[g.CAPTURED], "area": s["area"],
                                     "centroid_alpha": s["centroid_alpha"], "D": s["D"], "R_mean": s["R_mean"], "A": s["A"]})

    study(False)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    study(True)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    n_geo = len(c5["spins"]) * len(incs) * n_img
    out = {"metric": "run time of the shadow survey (BASELINE config C5)", "unit": "s", "value": ms * 1e-3, "n_gpus": 1,
           "higher_is_better": False, "data": "synthetic", "dtype": "f32",
           "config": {"workload": "99 images (11 spins x 9 inclinations), 1024 x 1024 pixels over +-10 M at r_obs = 1000 M, eq. (2) rule "
                                  "h = 1/32, xi monitor eps = 1e-3, cap 20000 steps",
                      "timer": "CUDA events around the whole survey (per spin: 9 x init, one integrate launch, 9 x (classify + shadow edge read "
                               "back)), after one warm-up pass"},
           "geodesics": n_geo, "geodesics_per_s": n_geo / (ms * 1e-3), "photon_steps": steps, "photon_steps_per_s": steps / (ms * 1e-3),
           "rays_bad_or_live": bad, "rows": rows}
    del big, views
    if emit:
        print(json.dumps(out), flush=True)
    return out


def launcher_command(args, argv, port=None):
    """`python bench.py --gpus N` started by hand (no torchrun environment): the command that re-runs this script as N
    ranks on this node, one per GPU, the way the driver launches it.  None if no re-launch is needed."""
    if args.gpus <= 1 or "WORLD_SIZE" in os.environ or args.impl == "reference":
        return None
    if port is None:
        import socket
        with socket.socket() as sock:
            sock.bind(("127.0.0.1", 0))
            port = sock.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def main():
    args = parse()
    cmd = launcher_command(args, sys.argv[1:])
    if cmd is not None:
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "INFO")          # NCCL's init log on stderr: the driver can count the ranks
        raise SystemExit(subprocess.call(cmd, env=env))
    if args.case == "projection" and args.impl != "reference":
        run_projection(args)
        return
    if args.case == "ring" and args.impl != "reference":
        run_ring(args)
        return
    if args.case == "survey" and args.impl != "reference":
        run_survey(args)
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gray(args)


if __name__ == "__main__":
    main()
