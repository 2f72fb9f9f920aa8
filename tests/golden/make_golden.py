#!/usr/bin/env python
"""Writes the stored expected values of the FULL-LENGTH parity runs (north_star: "after the stated number of steps",
PAPER.md:204 fixed step counts) for the configs whose oracle run is too long for the test suite:

    config 2: M = 36,  N = 2^18, 500 steps      config 3: M = 120, N = 2^18, 200 steps

Command (run once on a CPU box, from the repo root; ~30-45 min per config on 8 cores, ~8 GiB of RAM for config 3):

    python tests/golden/make_golden.py 2 3

and, for config 4 (M = 120, N = 2^22) on ITS OWN seeded, non-periodic field, a SHORT run of 2 steps (a whole oracle step
of that size takes ~2 min on 16 threads and the run needs ~115 GiB of RAM: E + six field buffers + the field):

    python tests/golden/make_golden.py 4:2 [output directory]     -> cfg4_2steps.npz (coarser sampling: ~1.3 MB)

This script imports ONLY `oracle/` (the CPU oracle) and `paper_1901_01895_b200/workloads.py` (seeded inputs and
parameters, no method arithmetic).  Nothing here comes from the CUDA path.  Output per config, `tests/golden/
cfg<id>_full.npz`:
    rows_dense   the rows sampled densely                         idx_dense   their sample indices (every 64th)
    dense        oracle output at [rows_dense, idx_dense]         idx_all     sample indices taken from EVERY row
    all          oracle output at [:, idx_all]                    norm2       sum |A|^2 of every output row
    meta         [cfg, M, N, steps]
tests/test_gpu_fullsize.py::test_full_length_matches_golden runs mmf_propagate for the full step count and compares
these samples element-wise (relative L2 over the stored samples of each row <= 1e-10) and the row energies.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle as orc  # noqa: E402
from paper_1901_01895_b200 import workloads  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
DENSE_STRIDE = 64      # every 64th sample of the densely sampled rows
ALL_STRIDE = 4096      # every 4096th sample (offset 37: not a tile border) of every row
ALL_OFFSET = 37


def dense_rows(R):
    """first, second, two in the middle (an x / y pair) and the last row"""
    return np.array(sorted({0, 1, R // 2, R // 2 + 1, R - 1}), dtype=np.int64)


def sample_indices(N):
    return np.arange(0, N, DENSE_STRIDE, dtype=np.int64), np.arange(ALL_OFFSET, N, ALL_STRIDE, dtype=np.int64)


def field_threaded(p):
    """p.field() with the rows generated side by side (workloads only; every row has its own seeded generator)."""
    from concurrent.futures import ThreadPoolExecutor
    A = np.empty((p.R, p.N), dtype=np.complex128)

    def one(r):
        A[r] = p.row(r)

    with ThreadPoolExecutor(max_workers=orc.default_threads()) as ex:
        list(ex.map(one, range(p.R)))
    return A


def make_short(cfg, steps, outdir):
    """`steps` oracle steps of config `cfg` at full size on its own field; sampled more coarsely than make()."""
    p = workloads.problem(cfg)
    need = (7 * p.R * p.N * 16 + p.M * p.N * 16) / 2 ** 30
    avail = [int(l.split()[1]) for l in open("/proc/meminfo") if l.startswith("MemAvailable")][0] / 2 ** 20
    print("cfg%d x %d steps: needs ~%.0f GiB, %.0f GiB available" % (cfg, steps, need, avail), flush=True)
    if avail < need + 16:
        raise SystemExit("not enough memory for the oracle at this size: refusing to start")
    A = field_threaded(p)
    t0 = time.perf_counter()
    out = orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, steps, inplace=True)
    dt = time.perf_counter() - t0
    rows = dense_rows(p.R)
    idx_d = np.arange(0, p.N, 1024, dtype=np.int64)
    idx_a = np.arange(ALL_OFFSET, p.N, 16384, dtype=np.int64)
    path = os.path.join(outdir, "cfg%d_%dsteps.npz" % (cfg, steps))
    np.savez(path, rows_dense=rows, idx_dense=idx_d, dense=out[np.ix_(rows, idx_d)], idx_all=idx_a,
             all=out[:, idx_a], norm2=np.sum(out.real ** 2 + out.imag ** 2, axis=1),
             meta=np.array([cfg, p.M, p.N, steps], dtype=np.int64))
    print("cfg%d: %d steps of %d x 2^%d in %.0f s on %d threads -> %s (%d bytes)" % (
        cfg, steps, p.R, p.N.bit_length() - 1, dt, orc.default_threads(), path, os.path.getsize(path)), flush=True)


def make(cfg):
    p = workloads.problem(cfg)
    A = p.field()
    t0 = time.perf_counter()
    out = orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, p.steps)
    dt = time.perf_counter() - t0
    rows = dense_rows(p.R)
    idx_d, idx_a = sample_indices(p.N)
    path = os.path.join(HERE, "cfg%d_full.npz" % cfg)
    np.savez(path, rows_dense=rows, idx_dense=idx_d, dense=out[np.ix_(rows, idx_d)], idx_all=idx_a,
             all=out[:, idx_a], norm2=np.sum(out.real ** 2 + out.imag ** 2, axis=1),
             meta=np.array([cfg, p.M, p.N, p.steps], dtype=np.int64))
    print("cfg%d: %d steps of %d x 2^%d in %.0f s on %d threads -> %s (%d bytes)" % (
        cfg, p.steps, p.R, p.N.bit_length() - 1, dt, orc.default_threads(), path, os.path.getsize(path)), flush=True)


if __name__ == "__main__":
    args = sys.argv[1:]
    if args and ":" in args[0]:
        c, st = (int(x) for x in args[0].split(":"))
        make_short(c, st, args[1] if len(args) > 1 else HERE)
    else:
        for c in (int(a) for a in args):
            make(c)
