"""Per-kernel counters of an `ncu --set full` capture of bench.py, as JSON for `profiles/` — bench.py's roofline
reads `traffic` (dram__bytes_read.sum + dram__bytes_write.sum per launch) and the fp64 thread-instruction count from
the file this writes, never from literals.

    python -m paper_1901_01895_b200.ncu_summary gpurun_out/<capture>.ncu-rep "<command that made it>" \
        > profiles/<round>_counters_cfg4.json

The capture must add the three fp64 op counters to the full set:
    ncu --set full --metrics smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,\
smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,smsp__sass_thread_inst_executed_op_dfma_pred_on.sum ...
The JSON is stamped with a hash of the kernel sources (csrc/*): bench.py emits null instead of stale counters when
the sources it runs differ from the ones profiled.  No arithmetic of the method lives here.
"""
import csv
import hashlib
import json
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")

NLT_MODES = ["plain", "s23", "final", "final_next", "rk4", "enter", "exit", "agrawal"]

METRICS = {
    "ms": ("gpu__time_duration.sum", 1e-6),                      # ns -> ms
    "dram_read_bytes": ("dram__bytes_read.sum", None),
    "dram_write_bytes": ("dram__bytes_write.sum", None),
    "dram_pct": ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", 1.0),
    "fp64_pipe_pct": ("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", 1.0),
    "lsu_data_pipe_pct": ("l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed", 1.0),
    "issue_pct": ("sm__inst_issued.avg.pct_of_peak_sustained_active", 1.0),
    "smem_wavefronts": ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", 1.0),
    "smem_bank_conflicts": ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", 1.0),
    "registers": ("launch__registers_per_thread", 1.0),
    "warp_inst": ("smsp__inst_executed.sum", 1.0),
    "dadd": ("smsp__sass_thread_inst_executed_op_dadd_pred_on.sum", 1.0),
    "dmul": ("smsp__sass_thread_inst_executed_op_dmul_pred_on.sum", 1.0),
    "dfma": ("smsp__sass_thread_inst_executed_op_dfma_pred_on.sum", 1.0),
    "sm_cycles": ("sm__cycles_elapsed.max", 1.0),
}
UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
              "ns": 1.0, "us": 1e3, "ms": 1e6, "s": 1e9, "nsecond": 1.0, "usecond": 1e3, "msecond": 1e6, "second": 1e9}


def source_hash():
    """sha256 over the kernel sources (file name + content, sorted) — identifies the build a capture belongs to."""
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh")) and name != "probes.cu":
            h.update(name.encode())
            with open(os.path.join(CSRC, name), "rb") as f:
                h.update(f.read())
    return h.hexdigest()


def kernel_class(name):
    """ncu's demangled kernel name -> the class name mmf_kernel_class_name() / bench.py use."""
    m = re.search(r"\b(k_\w+)<([^>]*)>", name)
    if not m:
        return None
    base, args = m.group(1), [int(x) for x in re.findall(r"-?\d+", re.sub(r"\((int|bool)\)", "", m.group(2)))]
    if base == "k_rows":
        return "k_rows"
    if base == "k_cols":
        return "k_cols<fwd>" if args[1] == 0 else "k_cols<inv>"
    if base == "k_nlt":
        return "k_nlm<%s>" % NLT_MODES[args[1]]
    if base == "k_nlg":
        return "k_nlg<%s>" % NLT_MODES[args[1]]
    return base


def stall_columns(hdr):
    return [i for i, h in enumerate(hdr) if h.startswith("smsp__pcsamp_warps_issue_stalled") and not h.endswith("not_issued")]


def summarise(rep):
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(out.splitlines()))
    hdr, units, data = rows[0], rows[1], rows[2:]
    ki = hdr.index("Kernel Name")
    stalls = stall_columns(hdr)
    per = {}
    for d in data:
        cls = kernel_class(d[ki])
        if cls is None:
            continue
        e = {}
        for key, (metric, scale) in METRICS.items():
            if metric not in hdr:
                continue
            i = hdr.index(metric)
            try:
                v = float(d[i].replace(",", ""))
            except ValueError:
                continue
            u = units[i]
            if key.endswith("_bytes"):
                v *= UNIT_SCALE.get(u, 1.0)
            elif key == "ms":
                v *= UNIT_SCALE.get(u, 1.0) * 1e-6
            e[key] = v
        tot = sum(float(d[i] or 0) for i in stalls) or 1.0
        top = sorted(((float(d[i] or 0) / tot * 100, hdr[i].replace("smsp__pcsamp_warps_issue_stalled_", "")) for i in stalls),
                     reverse=True)[:5]
        e["top_stalls_pct"] = {n: round(x, 1) for x, n in top}
        per.setdefault(cls, []).append(e)
    kernels = {}
    for cls, lst in per.items():
        avg = {}
        for key in lst[0]:
            if key == "top_stalls_pct":
                avg[key] = lst[0][key]
            else:
                vals = [x[key] for x in lst if key in x]
                avg[key] = sum(vals) / len(vals)
        avg["launches_captured"] = len(lst)
        if "dram_read_bytes" in avg:
            avg["traffic_bytes"] = avg["dram_read_bytes"] + avg["dram_write_bytes"]
        if all(k in avg for k in ("dadd", "dmul", "dfma")):
            avg["fp64_thread_inst"] = avg["dadd"] + avg["dmul"] + avg["dfma"]
        kernels[cls] = avg
    return kernels


def main():
    rep = sys.argv[1]
    command = sys.argv[2] if len(sys.argv) > 2 else ""
    print(json.dumps({"capture": os.path.basename(rep), "command": command, "source_sha256": source_hash(),
                      "per_launch_averages": True, "kernels": summarise(rep)}, indent=1, sort_keys=True))


if __name__ == "__main__":
    main()
