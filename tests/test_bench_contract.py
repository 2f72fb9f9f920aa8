"""bench.py's reference arm (the CPU oracle on a bounded sample; tier rule 4) prints ONE JSON line with the contract's
keys — checked here on the smallest config, where it takes a second.  The CUDA arm needs a GPU and is exercised by
the driver; its shard arguments (bench.py --shard) go through sharded.shard_arguments, tested in test_sharded_gloo.py."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*flags):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--cfg", "0", "--steps", "2",
                          "--warmup", "1"] + list(flags), capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_reference_arm_prints_the_contract_line():
    d = _run()
    assert d["impl"] == "reference" and d["metric"] == "rk4ip_field_sample_steps_per_s"
    assert d["unit"] == "field-sample-steps/s" and d["higher_is_better"] is True and d["dtype"] == "f64"
    assert d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] == 1 and d["vs_baseline"] is None
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["gpu_launches"] == 0
    assert abs(d["value"] - 4 * 4096 / (d["ms_per_step"] * 1e-3)) <= 1e-6 * d["value"]      # R N steps / time
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and "cfg0" in cb["sample"]
    e = d["e2e"]
    assert e["value"] == d["value"] and e["h2d_bytes_per_step"] == 0 and e["d2h_bytes_per_step"] == 0
    assert "workload" in d["config"] and "cfg0" in d["config"]["workload"]


def test_reference_arm_times_the_split_step_oracles_too():
    for method in ("ssfm", "agrawal"):
        d = _run("--method", method)
        assert d["config"]["method"] == method and d["value"] > 0


def test_gpus_n_starts_n_ranks_by_itself():
    """`python bench.py --gpus 2` without a torchrun environment must start 2 ranks (one per GPU on the box); here the
    --dry-run leg (gloo, no CUDA) checks the launcher and the aggregation: n_gpus = 2, units summed, time = max."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "4", "--cfg", "0",
                          "--dry-run"], capture_output=True, text=True, timeout=300, env=env, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout                      # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["dry_run"] and d["n_gpus"] == 2 and d["gpus_requested"] == 2
    assert d["units"] == 2 * 4 * 4096 * 4                   # 2 ranks x (R = 4 rows x N = 4096) x 4 steps
    assert abs(d["ms_per_step"] - 110.0) < 1e-9             # the slower rank's (synthetic) time
    assert abs(d["value"] - d["units"] / 0.44) < 1e-3
