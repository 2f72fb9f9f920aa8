#!/usr/bin/env python
"""bench.py — RK4IP field-sample-steps/s on B200 (BASELINE.json `metric`), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cfg 4] [--impl mmf|reference]

A "step" is one RK4IP step (Eq. 6a-6f: four exp(h/2 L) applications, four N evaluations and the
stage sums) over the whole 2M x N field of the workload.  Default workload: config 4 of BASELINE.json (M = 120
modes x 2 polarisations, N = 2^22; the configuration the >= 60 % roofline target is quoted on; it fits one B200).
`value` is measured with the field resident in HBM; `e2e` goes through mmf_propagate_host (C ABI, HOST buffer:
host->device copy, K steps, device->host copy inside the timed region).  N > 1: replicas only (DESIGN.md
"Multi-GPU") — every rank propagates its own fibre, no data-path collective; value = sum of units / max time.

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "rk4ip_field_sample_steps_per_s"
UNIT = "field-sample-steps/s"


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch, from the committed `ncu --set full` capture of this
# command on cfg4 (profiles/r1h_ncu_full_cfg4.md); other workloads have no capture: traffic = null.
NCU_TRAFFIC_CFG4 = {"k_rows": 74.32e9, "k_cols<fwd>": 65.62e9, "k_cols<inv>": 65.47e9, "k_nlm<s23>": 64.38e9,
                    "k_nlm<final_next>": 64.36e9}


def load_peaks():
    """HBM GB/s of MEASURED_PEAKS.json (driver-written), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def workload_string(p):
    return ("cfg%d: M=%d modes x 2 pol, N=2^%d fp64 complex, dt=%g ps, h=%g m, K=4 beta terms, kappa %dx%d; "
            "input: %s" % (p.cfg, p.M, p.N.bit_length() - 1, p.dt, p.h, p.M, p.M, p._c["signal"]))


def fill_field(p, out, nthreads):
    """Write the seeded input rows of problem p into the (2M, N) complex128 numpy array `out`."""
    from concurrent.futures import ThreadPoolExecutor

    def one(r):
        out[r] = p.row(r)

    with ThreadPoolExecutor(max_workers=max(1, nthreads)) as ex:
        list(ex.map(one, range(p.R)))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # "under load" = samples in the upper half of the observed power range
        thr = 0.5 * (min(pw) + max(pw))
        load = [s for s, w in zip(sm, pw) if w >= thr] or sm
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------- the CPU oracle leg
ORACLE_SAMPLE_LOGN = 14


def oracle_sample(cfg):
    """Bounded sample of config `cfg` for the CPU oracle: same M, dt, h, fibre parameters and input recipe, with the
    time window cut to N = 2^14 samples (cfg 4: 1/256 of the window; per-sample work is unchanged except that each
    transform has 14 instead of 22 butterfly levels, which FAVOURS the CPU figure)."""
    from paper_1901_01895_b200 import workloads
    logn = min(workloads.CONFIGS[cfg]["N"].bit_length() - 1, ORACLE_SAMPLE_LOGN)
    p = workloads.problem(cfg, N=1 << logn)
    return p, p.field()


def oracle_steps(p, A, steps, nthreads):
    from oracle import oracle as orc
    t0 = time.perf_counter()
    orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, steps, nthreads=nthreads)
    return time.perf_counter() - t0


def time_oracle(cfg, budget_s):
    """cpu_baseline leg: the oracle as it stands, all host cores, about `budget_s` seconds of work."""
    from oracle import oracle as orc
    orc.build()
    p, A = oracle_sample(cfg)
    nthreads = orc.default_threads()
    t1 = oracle_steps(p, A, 1, nthreads)
    steps = int(max(1, min(500, budget_s / max(t1, 1e-3))))
    dt = oracle_steps(p, A, steps, nthreads)
    sample = "cfg%d recipe with N cut to 2^%d (M=%d, %d rows), %d steps in %.1f s" % (
        cfg, p.N.bit_length() - 1, p.M, p.R, steps, dt)
    return p.R * p.N * steps / dt, nthreads, sample


def run_reference(args):
    """--impl reference: the reference arm of this tier is the CPU oracle (no GPU work, rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    from oracle import oracle as orc
    from paper_1901_01895_b200 import workloads
    orc.build()
    p, A = oracle_sample(args.cfg)
    nthreads = orc.default_threads()
    for _ in range(args.warmup):
        oracle_steps(p, A, 1, nthreads)
    tsum = 0.0
    for _ in range(args.steps):
        tsum += oracle_steps(p, A, 1, nthreads)
    value = p.R * p.N * args.steps / tsum
    sample = "each step = 1 RK4IP step of the cfg%d recipe with N cut to 2^%d (M=%d, %d rows)" % (
        args.cfg, p.N.bit_length() - 1, p.M, p.R)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tsum / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_string(workloads.problem(args.cfg)), "l2": "n/a (CPU oracle)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": nthreads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------- the CUDA leg
def run_mmf(args):
    import numpy as np
    import torch
    from paper_1901_01895_b200 import binding, replicas, workloads

    rank, local_rank, world = replicas.env_rank_world()
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group(backend="nccl", device_id=torch.device("cuda", local_rank))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    binding.lib()                                   # fail loudly if the CUDA library is missing
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)

    p = workloads.problem(args.cfg, M=args.modes, N=None if args.logn is None else 1 << args.logn)
    F = p.R * p.N * 16
    log("[bench] rank %d/%d: %s, field copy F = %.2f GiB" % (rank, world, workload_string(p), F / 2 ** 30))
    t0 = time.perf_counter()
    H = torch.empty((p.R, p.N), dtype=torch.complex128, pin_memory=True)        # host copy of the input (pinned)
    nthreads = max(1, len(os.sched_getaffinity(0)) // max(1, world))
    fill_field(p, H.numpy(), nthreads)
    log("[bench] input generated in %.1f s" % (time.perf_counter() - t0))
    X = torch.empty((p.R, p.N), dtype=torch.complex128, device=dev)
    X.copy_(H)
    if world > 1:                                    # replicas: a launch-power sweep, one power per rank
        X *= replicas.amplitude_scale(rank, world)
        H.copy_(X)
    plan = binding.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, device=dev)
    stream = torch.cuda.current_stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up (W untimed steps), then K timed steps, field resident in HBM ----
    advance = plan.propagate if args.method == "rk4ip" else plan.propagate_ssfm
    advance(X, args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    plan.set_timing(True)
    n0 = plan.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    advance(X, args.steps)
    e1.record(stream)
    barrier()
    launches = plan.launch_count() - n0
    ms = e0.elapsed_time(e1)
    kern = plan.get_timing()
    plan.set_timing(False)
    clocks = sampler.stop()
    _, ms, value = replicas.whole_job(p.R * p.N * args.steps, ms, dist, dev)
    assert bool(torch.isfinite(X.view(torch.float64)).all()), "propagated field is not finite"

    # ---- end to end: host buffer in, host buffer out, through the C ABI ----
    barrier()
    e0.record(stream)
    if args.method == "rk4ip":
        plan.propagate_host(H, X, args.steps)       # H2D copy, K steps, D2H copy, stream synchronised inside
    else:                                           # no host entry point for the split step: same copies by hand
        X.copy_(H, non_blocking=True)
        advance(X, args.steps)
        H.copy_(X, non_blocking=True)
    e1.record(stream)
    barrier()
    ms_e2e = e0.elapsed_time(e1)                    # device clock over the whole call
    _, ms_e2e, e2e_value = replicas.whole_job(p.R * p.N * args.steps, ms_e2e, dist, dev)

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel (largest summed device time in the timed region) ----
    peak, peak_src = load_peaks()
    full_cfg4 = args.cfg == 4 and args.modes is None and args.logn is None and args.method == "rk4ip"
    roof = None
    breakdown = []
    tot_kernel_ms = sum(k["total_ms"] for k in kern) or 1.0
    for k in kern:
        avg = k["total_ms"] / k["launches"]
        gbs = k["alg_bytes_per_launch"] / (avg * 1e-3) / 1e9
        breakdown.append({"kernel": k["name"], "launches": k["launches"], "avg_ms": round(avg, 4),
                          "share": round(k["total_ms"] / tot_kernel_ms, 4), "alg_GBps": round(gbs, 1)})
    if kern:
        top = max(kern, key=lambda k: k["total_ms"])
        avg = top["total_ms"] / top["launches"]
        ach = top["alg_bytes_per_launch"] / (avg * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": top["name"], "achieved": ach, "peak": peak, "unit": "GB/s",
                "frac": ach / peak, "traffic": NCU_TRAFFIC_CFG4.get(top["name"]) if full_cfg4 else None,
                "traffic_source": "profiles/r1h_ncu_full_cfg4.md" if full_cfg4 else None, "peak_source": peak_src,
                "alg_bytes_per_launch": top["alg_bytes_per_launch"], "avg_launch_ms": avg}
        if full_cfg4 and top["name"] == "k_rows":
            # second bound of the same kernel: fp64 issue.  Thread-level fp64 instructions of one launch from the
            # committed ncu capture (smsp__inst_executed x fp64 share, profiles/r1h_ncu_full_cfg4.md); peak = 64 per
            # clock per SM x 148 SMs (measured with a DADD / DMUL stream) at the clock seen under load.
            fp64_inst = 1.69e11
            clk = (clocks.get("sm_mhz") or 1965.0) * 1e6
            peak_i = 64.0 * 148 * clk
            roof["fp64_issue"] = {"achieved_Tinst_s": fp64_inst / (avg * 1e-3) / 1e12, "peak_Tinst_s": peak_i / 1e12,
                                  "frac": fp64_inst / (avg * 1e-3) / peak_i, "sm_mhz": clk / 1e6}
    # whole-step roofline: B_alg = 36 F (three-pass transforms) or 20 F (rows fit on chip)
    if args.method == "rk4ip":
        balg = (36 if p.N > 4096 else 20) * F
    else:                                           # two D on one buffer (3 passes x 2 F, or 2 F on chip) + 2 F
        balg = (14 if p.N > 4096 else 6) * F
    t_roof_ms = balg / (peak * 1e9) * 1e3
    step_roof = {"B_alg_bytes_per_step": balg, "hbm_time_ms": t_roof_ms, "frac": t_roof_ms / (ms / args.steps)}
    if args.method == "rk4ip" and p.N > 4096:      # this plan's own count: (6c)+(6d) in one pass -> 32 F
        step_roof["frac_of_32F_plan"] = (32 * F / (peak * 1e9) * 1e3) / (ms / args.steps)

    # ---- cuFFT (through torch.fft) beside the hand-written transforms: a reference point only, never on the path ----
    cufft = None
    if not args.no_cufft and world == 1:
        try:
            Ecf = torch.ones((p.M, 1, p.N), dtype=torch.complex128, device=dev)   # stands in for exp(h/2 L)/N
            Xv = X.view(p.M, 2, p.N)

            def d_cufft():
                S = torch.fft.fft(Xv, dim=2)
                S *= Ecf
                torch.fft.ifft(S, dim=2, out=Xv)

            d_cufft()
            torch.cuda.synchronize()
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0.record(stream)
            for _ in range(3):
                d_cufft()
            c1.record(stream)
            torch.cuda.synchronize()
            ms_cf = c0.elapsed_time(c1) / 3
            ours = sum(k["total_ms"] / k["launches"] for k in kern if k["name"] in ("k_cols<fwd>", "k_rows", "k_cols<inv>"))
            cufft = {"what": "one D = ifft(E * fft(x)) over the whole field with torch.fft (cuFFT, out of place + "
                             "elementwise multiply)", "ms_per_field": ms_cf,
                     "ours_ms_per_field": ours / 2 if p.N > 4096 else None}
            del Ecf
        except Exception as exc:                     # reference point only: never fail the bench on it
            cufft = {"unavailable": repr(exc)[:200]}

    # ---- the CPU oracle, timed on this box's host cores on a bounded sample ----
    cpu = None
    if not args.no_cpu:
        fss, cores, sample = time_oracle(args.cfg, budget_s=args.cpu_seconds)
        cpu = {"value": fss, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_string(p), "method": args.method, "l2": "field copy %.1f GiB >> 126 MB L2 (no flush needed)"
                       % (F / 2 ** 30) if F > 4 * 126e6 else "working set near/below L2 size: L2-resident",
                       "parallelism": "replicas x%d (launch-power sweep, no collective)" % world},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": F / args.steps,
                    "d2h_bytes_per_step": F / args.steps, "ms_per_call": ms_e2e,
                    "call": "mmf_propagate_host(nsteps=%d): one H2D + one D2H of F per call" % args.steps},
            "gpu_launches": launches, "roofline": roof, "step_roofline": step_roof, "kernels": breakdown, "cufft_reference": cufft,
            "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--cfg", type=int, default=4, help="BASELINE.json config id (default 4: M=120, N=2^22)")
    ap.add_argument("--impl", default="mmf", choices=["mmf", "reference"])
    ap.add_argument("--method", default="rk4ip", choices=["rk4ip", "ssfm"],
                    help="rk4ip (Eq. 6, the headline path) or ssfm (SSFM-RK4, the symmetric split step of Eq. 4)")
    ap.add_argument("--modes", type=int, default=None, help="override the config's mode count M (extra data points)")
    ap.add_argument("--logn", type=int, default=None, help="override the config's N = 2^logn (extra data points)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT reference point")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_mmf(args)


if __name__ == "__main__":
    sys.exit(main())
