#!/usr/bin/env python
"""Accuracy versus step size of the three schemes the paper names — RK4IP (Eq. 6), SSFM-RK4 and SSFM-Agrawal (Eq. 4,
PAPER.md:58-63) — on config 0 (M = 2 modes, N = 2^12, its fibre parameters and QPSK recipe) over 20 km at 100 x the
launch power, written to tests/golden/stepsize_table.md.  (Config 0 rather than a shrunken config 2: with 60 WDM
channels the dispersion phase across the band is thousands of radians per step and none of the schemes is in its
asymptotic regime at affordable step sizes — the orders of accuracy would not show.)  It reproduces the paper's reason for RK4IP: "The RK4IP allows
more than doubled step-sizes h".

    python tests/golden/make_stepsize_table.py          # ~3 min on 8 cores

Imports ONLY oracle/ and paper_1901_01895_b200/workloads.py (seeded inputs, no method arithmetic).  The error of a run
is the largest per-field relative L2 distance to an RK4IP run 8 x finer than the finest row (h = 3.9 m).
tests/test_oracle_ssfm_pins.py::test_stepsize_table_claim re-derives two rows and checks the claim.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle as orc  # noqa: E402
from paper_1901_01895_b200 import workloads  # noqa: E402

LENGTH_M = 20000.0
STEPS = (10, 20, 40, 80, 160, 320, 640)     # h = 2000 ... 31.25 m
POWER_SCALE = 10.0                           # 100 x the config's launch power: a nonlinear phase of a few rad over 20 km
REF_FACTOR = 8                               # the reference run has REF_FACTOR x the steps of the finest row


def setup():
    p = workloads.problem(0)
    return p, p.field() * POWER_SCALE


def errors(p, A, ref, steps):
    out = {}
    h = LENGTH_M / steps
    runs = {"RK4IP": lambda: orc.rk4ip(A, p.dt, h, p.alpha, p.beta, p.gamma, p.kappa, steps),
            "SSFM-RK4": lambda: orc.ssfm_rk4(A, p.dt, h, p.alpha, p.beta, p.gamma, p.kappa, steps),
            "SSFM-Agrawal (2 it.)": lambda: orc.ssfm_agrawal(A, p.dt, h, p.alpha, p.beta, p.gamma, p.kappa, steps, niter=2)}
    for name, f in runs.items():
        out[name] = float(workloads.rel_l2_per_field(f(), ref).max())
    return out


def reference(p, A, n=None):
    n = REF_FACTOR * STEPS[-1] if n is None else n
    return orc.rk4ip(A, p.dt, LENGTH_M / n, p.alpha, p.beta, p.gamma, p.kappa, n)


def step_for_accuracy(hs, errs, target):
    """largest h with error <= target, by log-log interpolation between the bracketing rows"""
    for i in range(len(hs) - 1):
        if errs[i] > target >= errs[i + 1]:
            s = np.log(errs[i] / errs[i + 1]) / np.log(hs[i] / hs[i + 1])
            return float(hs[i + 1] * (target / errs[i + 1]) ** (1.0 / s))
    return None


def main():
    p, A = setup()
    ref = reference(p, A)
    rows = [(LENGTH_M / n, errors(p, A, ref, n)) for n in STEPS]
    names = list(rows[0][1])
    lines = ["# Error versus step size: RK4IP, SSFM-RK4, SSFM-Agrawal (oracle only)", "",
             "Written by `python tests/golden/make_stepsize_table.py` (calls only `oracle/` and `workloads.py`).",
             "Workload: config 0 (M = 2, N = 2^12, dt = 1 ps), 20 km, amplitudes x %g; error = max over fields of"
             % POWER_SCALE, "the relative L2 distance to RK4IP at h = %.4g m." % (LENGTH_M / (REF_FACTOR * STEPS[-1])), "",
             "| h [m] | steps | " + " | ".join(names) + " |", "|---|---|" + "---|" * len(names)]
    for h, e in rows:
        lines.append("| %.5g | %d | " % (h, round(LENGTH_M / h)) + " | ".join("%.3e" % e[n] for n in names) + " |")
    hs = [h for h, _ in rows]
    lines += ["", "Step size that reaches a given error (log-log interpolation), and the ratio to RK4IP's:", "",
              "| target error | " + " | ".join("h %s [m]" % n for n in names) + " | RK4IP / SSFM-RK4 | RK4IP / SSFM-Agrawal |",
              "|---|" + "---|" * (len(names) + 2)]
    for target in (1e-3, 1e-4):
        hh = [step_for_accuracy(hs, [e[n] for _, e in rows], target) for n in names]
        cells = ["%.4g" % x if x else "outside the table" for x in hh]
        ratios = ["%.2f" % (hh[0] / x) if (hh[0] and x) else "-" for x in hh[1:]]
        lines.append("| %.0e | " % target + " | ".join(cells) + " | " + " | ".join(ratios) + " |")
    lines += ["", "PAPER.md:113: \"The RK4IP allows more than doubled step-sizes h\" — the ratios above."]
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "stepsize_table.md")
    with open(path, "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
