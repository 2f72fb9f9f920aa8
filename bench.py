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


def load_counters(cfg):
    """Per-kernel ncu counters (DRAM traffic, fp64 thread instructions per launch) of the newest committed
    `ncu --set full` capture of this command: profiles/r*_counters_cfg<cfg>.json, written by
    paper_1901_01895_b200/ncu_summary.py.  Returns (kernels, file, stale): stale = the kernel sources have changed since
    the capture (then the numbers are NOT reported: traffic = null)."""
    import glob
    from paper_1901_01895_b200 import ncu_summary
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_counters_cfg%d.json" % cfg)))
    if not files:
        return {}, None, False
    with open(files[-1]) as f:
        d = json.load(f)
    return d.get("kernels", {}), os.path.relpath(files[-1], ROOT), d.get("source_sha256") != ncu_summary.source_hash()


def load_peaks():
    """HBM GB/s of MEASURED_PEAKS.json (driver-written), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def load_fp64_peak(sms):
    """fp64 peak [TFLOP/s]: the best DFMA / DMMA rate `bench.py --probes` measured (newest profiles/r*_probes.json),
    else derived: 64 DFMA per clock per SM x 2 flop x SM count x 1.965 GHz."""
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_probes.json")))
    if files:
        try:
            with open(files[-1]) as f:
                d = json.load(f)
            return max(e["TFLOP_s"] for e in d["probes"]["fp64"]), "measured (%s)" % os.path.relpath(files[-1], ROOT)
        except Exception:
            pass
    return 64 * 2 * sms * 1.965e9 / 1e12, "derived (64 DFMA/clk/SM x SMs x 1.965 GHz)"


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


def oracle_steps(p, A, steps, nthreads, method="rk4ip"):
    from oracle import oracle as orc
    fn = {"rk4ip": orc.rk4ip, "ssfm": orc.ssfm_rk4, "agrawal": orc.ssfm_agrawal}[method]
    t0 = time.perf_counter()
    fn(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, steps, nthreads=nthreads)
    return time.perf_counter() - t0


def host_description():
    """CPU model string and available RAM of the box the oracle is timed on."""
    model, avail = "unknown", None
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable"):
                    avail = round(int(line.split()[1]) / 2 ** 20, 1)
                    break
    except OSError:
        pass
    return model, avail


def time_oracle(cfg, budget_s, method="rk4ip"):
    """cpu_baseline leg: the oracle as it stands (UNOPTIMISED: textbook radix-2 transform, -O2, stage sums on one
    thread), all host cores, about `budget_s` seconds of work; plus the single-core figure on configs 0 and 1."""
    from oracle import oracle as orc
    from paper_1901_01895_b200 import workloads
    orc.build()
    p, A = oracle_sample(cfg)
    nthreads = orc.default_threads()
    t1 = oracle_steps(p, A, 1, nthreads, method)
    steps = int(max(1, min(500, budget_s / max(t1, 1e-3))))
    dt = oracle_steps(p, A, steps, nthreads, method)
    sample = "cfg%d recipe with N cut to 2^%d (M=%d, %d rows), %d %s steps in %.1f s" % (
        cfg, p.N.bit_length() - 1, p.M, p.R, steps, method, dt)
    single = {}
    for c, st in ((0, 20), (1, 2)):
        q = workloads.problem(c)
        ts = oracle_steps(q, q.field(), st, 1, method)
        single["cfg%d" % c] = q.R * q.N * st / ts
    return p.R * p.N * steps / dt, nthreads, sample, single


def run_reference(args):
    """--impl reference: the reference arm of this tier is the CPU oracle (no GPU work, rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    from oracle import oracle as orc
    from paper_1901_01895_b200 import workloads
    orc.build()
    p, A = oracle_sample(args.cfg)
    nthreads = orc.default_threads()
    method = args.method
    for _ in range(args.warmup):
        oracle_steps(p, A, 1, nthreads, method)
    tsum = 0.0
    for _ in range(args.steps):
        tsum += oracle_steps(p, A, 1, nthreads, method)
    value = p.R * p.N * args.steps / tsum
    sample = "each step = 1 %s step of the cfg%d recipe with N cut to 2^%d (M=%d, %d rows)" % (
        method, args.cfg, p.N.bit_length() - 1, p.M, p.R)
    model, avail = host_description()
    full = workloads.problem(args.cfg)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tsum / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_string(full) + (
                           " -- THIS ARM RAN A BOUNDED SAMPLE OF IT: N cut from 2^%d to 2^%d, everything else unchanged"
                           % (full.N.bit_length() - 1, p.N.bit_length() - 1) if p.N != full.N else ""),
                       "workload_run": workload_string(p), "method": method, "l2": "n/a (CPU oracle)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": nthreads, "kind": "oracle",
                             "note": "unoptimised test infrastructure (textbook radix-2, -O2)", "sample": sample, "cpu_model": model, "mem_available_GiB": avail},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------ measurement probes
def run_probes(args):
    """--probes: the denominators DESIGN.md §6 quotes, measured live through the C ABI (mmf_probe_fp64,
    mmf_probe_tma_copy): fp64 issue peaks of the plain and the tensor (DMMA) path, and what a pure TMA copy through
    the product kernels' ring reaches with each kernel's access pattern on a config-4 sized buffer."""
    import torch
    from paper_1901_01895_b200 import binding
    assert torch.cuda.is_available()
    binding.lib()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    sampler = ClockSampler(0)
    sampler.start()
    fp = []
    names = ["DADD x=x+y", "DMUL x=x*y", "DFMA x=fma(y,z,x) (3 distinct regs)", "DFMA x=fma(x,y,y) (2 distinct regs)",
             "add/sub butterfly (2 DADD)", "DMMA m8n8k4 (4 chains per warp)"]
    for kind, name in enumerate(names):
        for threads in (512, 1024):
            ms, n = binding.probe_fp64(kind, threads=threads, iters=4000)
            e = {"kind": name, "threads_per_sm": threads, "ms": round(ms, 3)}
            if kind == 5:
                e["TFLOP_s"] = round(n * 512 / (ms * 1e-3) / 1e12, 2)
                e["warp_inst_per_s_per_sm"] = n / (ms * 1e-3) / sms
            else:
                e["thread_inst_per_s_per_sm"] = n / (ms * 1e-3) / sms
                e["TFLOP_s"] = round(n * (2 if kind in (2, 3) else 1) / (ms * 1e-3) / 1e12, 2)
            fp.append(e)
    clocks = sampler.stop()
    clk = (clocks.get("sm_mhz") or 1965.0) * 1e6
    for e in fp:
        if "thread_inst_per_s_per_sm" in e:
            e["thread_inst_per_clk_per_sm"] = round(e.pop("thread_inst_per_s_per_sm") / clk, 1)
        else:
            e["clk_per_dmma_per_sm"] = round(clk / e.pop("warp_inst_per_s_per_sm"), 2)
    # on-chip data paths of a 4096-point tile (16 complex values per thread): bytes per clock per SM where the kind moves
    # a fixed 128 B per thread and operation, clock64 ticks per operation (per warp stage) otherwise
    onchip = []
    oc_names = ["tcgen05.ld 32x32b.x32 + wait", "tcgen05.st 32x32b.x32", "LDS.128 x 8", "SHFL.BFLY b32 x 32",
                "tensor-memory trip, forward (st 32x32b, ld 16x256b)", "tensor-memory trip, reverse (st 16x256b, ld 32x32b)",
                "warp-local exchange through shared memory", "group-wide exchange through shared memory (256 threads)",
                "radix-16 stage, registers only", "radix-16 stage + 15 twiddles from shared memory"]
    for kind, name in enumerate(oc_names):
        for threads in ((256, 512) if kind == 7 else (32, 256, 512)):
            ms, clk_op = binding.probe_onchip(kind, threads=threads, iters=2000)
            e = {"kind": name, "threads_per_sm": threads, "clk_per_op": round(clk_op, 1)}
            if kind < 4:
                e["bytes_per_clk_per_sm"] = round(128.0 * threads / clk_op, 1)
            onchip.append(e)
    R, N, N1, N2 = 240, 1 << 22, 1 << 10, 1 << 12
    buf = torch.zeros(R * N * 16, dtype=torch.uint8, device=dev)
    # (name, dim0 [doubles], dim1 [rows], stride [B], box0, box1, nbox, nct_log, c0_mul, c1_mul, ntiles, slots, bulk)
    cases = [
        ("contiguous 64 KiB tiles (cp.async.bulk; pass B, natural order)", 0, 0, 0, 8192, 1, 1, 0, 0, 0, R * N // 4096, 3, 1),
        ("64 B segments at 64 KiB pitch, 1024 rows per tile (passes A/C, natural order)",
         2 * N2, R * N1, N2 * 16, 8, 256, 4, 10, 8, 1024, R * N2 // 4, 3, 0),
        ("64 B segments at 256 B pitch inside a contiguous block (passes A/C, blocked order WB=16)",
         32, R * (N2 // 16) * N1, 256, 8, 256, 4, 2, 8, 1024, R * N2 // 4, 3, 0),
        ("64 B segments at 128 B pitch (passes A/C, WB=8)", 16, R * (N2 // 8) * N1, 128, 8, 256, 4, 1, 8, 1024, R * N2 // 4, 3, 0),
        ("64 B segments at 1 KiB pitch (passes A/C, WB=64)", 128, R * (N2 // 64) * N1, 1024, 8, 256, 4, 4, 8, 1024, R * N2 // 4, 3, 0),
        ("256 B segments at 256 KiB pitch (pass B, blocked order WB=16)",
         2 * N1 * 16, R * (N2 // 16), N1 * 16 * 16, 32, 256, 1, 10, 32, 256, R * N1, 3, 0),
        ("128 B segments at 128 KiB pitch (pass B, WB=8)", 2 * N1 * 8, R * (N2 // 8), N1 * 8 * 16, 16, 256, 2, 10, 16, 512, R * N1, 3, 0),
        ("128 B segments at 64 MiB pitch, 240 rows per tile (nonlinear kernels, 8-sample tile)",
         2 * N, R, N * 16, 16, R, 1, 30, 16, 0, N // 8, 3, 0),
        ("same, 6 slots", 2 * N, R, N * 16, 16, R, 1, 30, 16, 0, N // 8, 6, 0),
        ("256 B segments at 64 MiB pitch, 240 rows per tile (16-sample tile)", 2 * N, R, N * 16, 32, R, 1, 30, 32, 0, N // 16, 3, 0),
    ]
    tma = []
    for c in cases:
        name, d0, d1, st, b0, b1, nbox, ncl, c0m, c1m, nt, slots, bulk = c
        ms, by = binding.probe_tma_copy(buf, d0, d1, st, b0, b1, nbox, ncl, c0m, c1m, nt, slots=slots, bulk=bulk, reps=3)
        tma.append({"pattern": name, "tile_bytes": nbox * b0 * b1 * 8, "slots": slots, "ms": round(ms, 3),
                    "GB_s": round(by / (ms * 1e-3) / 1e9, 0), "GB_moved": round(by / 1e9, 1)})
    peak, src = load_peaks()
    print(json.dumps({"probes": {"fp64": fp, "onchip": onchip, "tma_copy": tma}, "sms": sms, "clocks_during_fp64": clocks,
                      "hbm_peak_GB_s": peak, "hbm_peak_source": src}), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ N > 1 launcher
def relaunch_one_rank_per_gpu(args):
    """`python bench.py --gpus N` started plainly (no torchrun environment): start N ranks, one per GPU, the way the
    driver's multi-GPU command does (PAPER.md:164-168: one device per process; :186: one 8-GPU node) and hand back
    their exit code.  Rank 0 of the children prints the one JSON line with n_gpus = N.  The environment is passed on
    untouched (NCCL_DEBUG in particular: whatever the caller set stays set)."""
    import socket
    import subprocess
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    log("[bench] --gpus %d without a torchrun environment: starting %s" % (args.gpus, " ".join(cmd)))
    return subprocess.call(cmd)


def run_dry(args):
    """--dry-run: everything of the N-rank path that needs no GPU.  Rendezvous over gloo, then replicas.whole_job (sum of
    the units, max of the per-rank times) on SYNTHETIC per-rank times (100 ms per step on rank 0, 10 % more on every
    further rank), so that a test can check the aggregated line.  Not a measurement; the line says so."""
    from paper_1901_01895_b200 import replicas, workloads
    rank, _, world = replicas.env_rank_world()
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group(backend="gloo")
        dist.barrier()
    p = workloads.problem(args.cfg)
    ms_local = 100.0 * args.steps * (1.0 + 0.1 * rank)
    units, ms, value = replicas.whole_job(p.R * p.N * args.steps, ms_local, dist, None)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"dry_run": True, "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
                          "gpus_requested": args.gpus, "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": ms / args.steps, "units": units, "scaling": "weak", "data": "none (dry run)",
                          "config": {"workload": workload_string(p), "parallelism": "replicas x%d" % world}}), flush=True)
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
    general = args.kappa == "general"
    shard = None
    if args.shard:
        # row shards: this rank keeps modes mode0 .. mode0 + m - 1 and all-gathers the mode powers
        from paper_1901_01895_b200 import sharded
        assert args.method == "rk4ip" and not general, "--shard: rk4ip with the Manakov kappa"
        mode0, m, beta_l, kappa_rows = sharded.shard_arguments(p.beta, p.kappa, rank, world)
        H = H[2 * mode0:2 * (mode0 + m)]
        shard = sharded.CudaShardStages(p.M, mode0, p.N, p.dt, p.h, p.alpha, beta_l, p.gamma, kappa_rows, device=dev,
                                        chunks=args.shard_chunks)
    X = torch.empty(tuple(H.shape), dtype=torch.complex128, device=dev)
    X.copy_(H)
    if world > 1 and shard is None:                  # replicas: a launch-power sweep, one power per rank
        X *= replicas.amplitude_scale(rank, world)
        H.copy_(X)
    kappa = p.kappa_general() if general else p.kappa_grouped()[0] if args.kappa == "grouped" else p.kappa
    plan = shard.plan if shard is not None else binding.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, kappa, device=dev,
                                                              general=general)
    stream = torch.cuda.current_stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up (W untimed steps), then K timed steps, field resident in HBM ----
    advance = {"rk4ip": plan.propagate, "ssfm": plan.propagate_ssfm,
               "agrawal": lambda X_, n_: plan.propagate_ssfm_agrawal(X_, n_, niter=args.niter)}[args.method]
    if shard is not None:
        def advance(X_, n_):
            sharded.propagate(shard, X_, n_, lambda c: sharded.all_gather_rows(shard.P_all[c], shard.mode0, shard.M_local, dist,
                                                                             async_op=world > 1))
    advance(X, args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    # Per-launch CUDA events bracket every kernel of the timed region (the roofline's launch durations) — except for
    # the small configs, whose step body replays from a CUDA graph (mmf_api.cu): there the events would force the
    # launch-by-launch path and slow the very thing being measured, so the breakdown comes from a second, untimed pass.
    events_in_region = F > (64 << 20)
    plan.set_timing(events_in_region)
    n0 = plan.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    advance(X, args.steps)
    e1.record(stream)
    barrier()
    launches = plan.launch_count() - n0
    ms = e0.elapsed_time(e1)
    if not events_in_region:
        plan.set_timing(True)
        advance(X, min(args.steps, 20))
        torch.cuda.synchronize()
    kern = plan.get_timing()
    plan.set_timing(False)
    clocks = sampler.stop()
    # A second device-timed figure with the per-launch events OFF: that is how a caller runs the library (programmatic
    # dependent launch on, prologues overlapping the predecessor's tail).  The headline above keeps the events, because
    # the roofline's launch durations must come from the timed region itself.
    ms_product = value_product = None
    if events_in_region:
        barrier()
        e0.record(stream)
        advance(X, args.steps)
        e1.record(stream)
        barrier()
        _, ms_product, value_product = replicas.whole_job(X.shape[0] * p.N * args.steps, e0.elapsed_time(e1), dist, dev)
    _, ms, value = replicas.whole_job(X.shape[0] * p.N * args.steps, ms, dist, dev)
    assert bool(torch.isfinite(X.view(torch.float64)).all()), "propagated field is not finite"

    # ---- end to end: host buffers in, host buffers out, through the C ABI ----
    # (a) one field per call (mmf_propagate_host): H2D, K steps, D2H, all serial — one field cannot hide its copies;
    # (b) a stream of B fields per call (mmf_propagate_host_batch, e.g. a launch-power sweep): field i + 1 goes in and
    #     field i - 1 comes out while field i propagates.  (a) is e2e.value in every round; (b) is reported as e2e.batched.
    barrier()
    e0.record(stream)
    if args.method == "rk4ip" and shard is None:
        plan.propagate_host(H, X, args.steps)       # H2D copy, K steps, D2H copy, stream synchronised inside
    else:                                           # no host entry point for the split steps: same copies by hand
        X.copy_(H, non_blocking=True)
        advance(X, args.steps)
        H.copy_(X, non_blocking=True)
    e1.record(stream)
    barrier()
    ms_single = e0.elapsed_time(e1)                 # device clock over the whole call
    _, ms_single, single_value = replicas.whole_job(X.shape[0] * p.N * args.steps, ms_single, dist, dev)
    nbatch, ms_e2e, e2e_value = 1, ms_single, single_value
    if args.method == "rk4ip" and args.e2e_batch > 1 and shard is None:
        _, avail = host_description()
        free_dev = torch.cuda.mem_get_info(dev)[0]
        nbatch = args.e2e_batch
        while nbatch > 1 and ((avail or 0) * 2 ** 30 < (nbatch - 1) * F * world + (16 << 30)):
            nbatch -= 1
        if free_dev < F + (2 << 30):
            nbatch = 1
        if nbatch > 1:
            hosts = [H] + [torch.empty((p.R, p.N), dtype=torch.complex128, pin_memory=True) for _ in range(nbatch - 1)]
            for Hx in hosts[1:]:
                Hx.copy_(H)
            X2 = torch.empty_like(X)
            barrier()
            e0.record(stream)
            plan.propagate_host_batch(hosts, X, X2, args.steps)
            e1.record(stream)
            barrier()
            ms_e2e = e0.elapsed_time(e1)
            _, ms_e2e, e2e_value = replicas.whole_job(nbatch * p.R * p.N * args.steps, ms_e2e, dist, dev)
            del X2, hosts

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel (largest summed device time in the timed region) ----
    peak, peak_src = load_peaks()
    full_cfg = args.modes is None and args.logn is None and args.method == "rk4ip" and not general and shard is None
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
        counters, cfile, stale = load_counters(args.cfg) if full_cfg else ({}, None, False)
        ctr = {} if stale else counters.get(top["name"], {})
        roof = {"bound": "hbm", "kernel": top["name"], "achieved": ach, "peak": peak, "unit": "GB/s",
                "frac": ach / peak, "traffic": ctr.get("traffic_bytes"),
                "traffic_source": (cfile + (" (STALE: kernel sources changed since the capture; not reported)" if stale else ""))
                if cfile else None, "peak_source": peak_src,
                "alg_bytes_per_launch": top["alg_bytes_per_launch"], "avg_launch_ms": avg}
        if ctr.get("fp64_thread_inst"):
            # second bound of the same kernel: fp64 issue.  Thread-level fp64 instructions of one launch from the
            # committed capture (dadd + dmul + dfma counters); peak = 64 per clock per SM x the SM count
            # (profiles/r2_probes.md: measured with DADD / DMUL streams) at the clock seen under load.
            clk = (clocks.get("sm_mhz") or 1965.0) * 1e6
            peak_i = 64.0 * torch.cuda.get_device_properties(dev).multi_processor_count * clk
            roof["fp64_issue"] = {"thread_inst_per_launch": ctr["fp64_thread_inst"],
                                  "achieved_Tinst_s": ctr["fp64_thread_inst"] / (avg * 1e-3) / 1e12,
                                  "peak_Tinst_s": peak_i / 1e12, "frac": ctr["fp64_thread_inst"] / (avg * 1e-3) / peak_i,
                                  "sm_mhz": clk / 1e6}
    fp64_peak, fp64_src = load_fp64_peak(torch.cuda.get_device_properties(dev).multi_processor_count)
    if general and kern:
        # the general contraction is 2 (2M)^2 flop per sample per evaluation: its kernels are bound by the fp64 (tensor)
        # pipe, so the dominant one reports BOTH bounds (k_rows is co-limited by HBM and fp64 issue)
        nlg = [k for k in kern if k["name"].startswith("k_nlg")]
        if nlg:
            topg = max(nlg, key=lambda k: k["total_ms"])
            avg = topg["total_ms"] / topg["launches"]
            flops = 2.0 * (2 * p.M) ** 2 * p.N
            ach = flops / (avg * 1e-3) / 1e12
            gb = topg["alg_bytes_per_launch"] / (avg * 1e-3) / 1e9
            roof = {"bound": "alu", "kernel": topg["name"], "achieved": ach, "peak": fp64_peak, "unit": "TFLOP/s",
                    "frac": ach / fp64_peak, "traffic": None, "peak_source": fp64_src, "flop_per_launch": flops,
                    "avg_launch_ms": avg, "hbm": {"achieved": gb, "peak": peak, "unit": "GB/s", "frac": gb / peak,
                                                  "alg_bytes_per_launch": topg["alg_bytes_per_launch"]}}
    # whole-step roofline: B_alg = 36 F (three-pass transforms) or 20 F (rows fit on chip)
    if shard is not None:
        # per rank (its rows: F / world): transforms 24 F_r (8 on chip); powers kernels read 6 F_r and write 4 x F_r / 4;
        # apply kernels 13 F_r (four-buffer plan, one N per pass) and read the gathered powers 4 x world x F_r / 4
        balg = ((24 if p.N > 4096 else 8) + 20 + world) * F / world
    elif args.method == "rk4ip":
        balg = (36 if p.N > 4096 else 20) * F
    elif args.method == "agrawal":                  # (1 + niter) D on one buffer + S0 (1.25 F), IT1 (2.25 F), ITJ (3.25 F)
        balg = ((1 + args.niter) * (6 if p.N > 4096 else 2) + 3.5 + 3.25 * (args.niter - 1)) * F
    else:                                           # two D on one buffer (3 passes x 2 F, or 2 F on chip) + 2 F
        balg = (14 if p.N > 4096 else 6) * F
    t_roof_ms = balg / (peak * 1e9) * 1e3
    step_roof = {"B_alg_bytes_per_step": balg, "hbm_time_ms": t_roof_ms, "frac": t_roof_ms / (ms / args.steps)}
    if general:   # the slower of the step's bytes at HBM bandwidth and its fp64 flops at peak (north_star)
        t_alu_ms = 4 * 2.0 * (2 * p.M) ** 2 * p.N / (fp64_peak * 1e12) * 1e3
        step_roof.update({"alu_time_ms": t_alu_ms, "fp64_peak_TFLOP_s": fp64_peak,
                          "frac": max(t_roof_ms, t_alu_ms) / (ms / args.steps)})
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
        fss, cores, sample, single = time_oracle(args.cfg, budget_s=args.cpu_seconds,
                                                 method=args.method)
        model, avail = host_description()
        cpu = {"value": fss, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
               "note": "the oracle is unoptimised test infrastructure (textbook radix-2, -O2): a baseline, not a target",
               "single_core": single, "cpu_model": model, "mem_available_GiB": avail}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong" if shard is not None else "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_string(p) + (" [general 2M x 2M kappa]" if general else "") + (
                           " [mode-group kappa: %d distinct rows]" % plan.groups() if args.kappa == "grouped" else ""),
                       "method": args.method, "kappa": args.kappa, "l2": "field copy %.1f GiB >> 126 MB L2 (no flush needed)"
                       % (F / 2 ** 30) if F > 4 * 126e6 else "working set near/below L2 size: L2-resident",
                       "parallelism": ("row shards x%d (PAPER.md:99-168: whole rows per rank, all-gather of the mode powers 4x per "
                                       "step, NCCL)" % world) if shard is not None else
                                      "replicas x%d (launch-power sweep, no collective)" % world},
            "clocks": clocks,
            # e2e.value is the SINGLE-FIELD call in every round (round 1's definition: comparable across BENCH_rNN);
            # the overlapped stream of several fields is a different workload and sits under its own key.
            "e2e": {"value": single_value, "unit": UNIT, "h2d_bytes_per_step": F / args.steps,
                    "d2h_bytes_per_step": F / args.steps, "ms_per_call": ms_single, "fields_per_call": 1,
                    "call": "mmf_propagate_host(nsteps=%d): one H2D + one D2H of F per call, serial with the propagation"
                            % args.steps,
                    "batched": ({"value": e2e_value, "unit": UNIT, "ms_per_call": ms_e2e, "fields_per_call": nbatch,
                                 "call": "mmf_propagate_host_batch(nfields=%d, nsteps=%d): every field one H2D + one D2H "
                                         "of F, copies of neighbouring fields overlap the propagation"
                                         % (nbatch, args.steps)} if nbatch > 1 else None)},
            "as_called": ({"ms_per_step": ms_product / args.steps,
                           "value": value_product, "unit": UNIT,
                           "what": "the same K steps once more with the per-launch timing events off (programmatic "
                                   "dependent launch on): the step time a caller of mmf_propagate sees"}
                          if ms_product else None),
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
    ap.add_argument("--method", default="rk4ip", choices=["rk4ip", "ssfm", "agrawal"],
                    help="rk4ip (Eq. 6, the headline path), ssfm (SSFM-RK4) or agrawal (SSFM-Agrawal): the symmetric "
                         "split step of Eq. 4 with a Runge-Kutta resp. an iterative nonlinear part")
    ap.add_argument("--niter", type=int, default=2, help="iterations per step of --method agrawal")
    ap.add_argument("--kappa", default="manakov", choices=["manakov", "general", "grouped"],
                    help="manakov: kappa [M][M] of Eq. 1 (the headline path); general: the paper's [2M][2M] per-polarisation "
                         "matrix (PAPER.md:176; rk4ip only)")
    ap.add_argument("--shard", action="store_true",
                    help="row-sharded path (SURVEY.md NEXT-3): every rank propagates M / world modes and all-gathers the mode "
                         "powers; with one GPU it measures the split kernels alone")
    ap.add_argument("--shard-chunks", type=int, default=1,
                    help="--shard: time chunks per evaluation of N (the gather of one chunk overlaps the kernels of the next)")
    ap.add_argument("--modes", type=int, default=None, help="override the config's mode count M (extra data points)")
    ap.add_argument("--logn", type=int, default=None, help="override the config's N = 2^logn (extra data points)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT reference point")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--e2e-batch", type=int, default=3,
                    help="host fields per mmf_propagate_host_batch call of the end-to-end leg (1: single-field call only)")
    ap.add_argument("--probes", action="store_true",
                    help="measure the fp64 issue peaks and the TMA access-pattern ceilings instead of the benchmark")
    ap.add_argument("--dry-run", action="store_true",
                    help="launcher check without CUDA: start the ranks (gloo), run the barrier / max-over-ranks bookkeeping "
                         "of the timing contract on stated synthetic per-rank times, print the aggregated line")
    args = ap.parse_args()
    if args.probes:
        return run_probes(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return relaunch_one_rank_per_gpu(args)
    if args.dry_run:
        return run_dry(args)
    return run_mmf(args)


if __name__ == "__main__":
    sys.exit(main())
