"""Row-sharded RK4IP: the N > 1 path on CPU, world_size 2, gloo.

The driver under test is the product's (paper_1901_01895_b200/sharded.py: mode partition, step sequence, all-gather
of the mode powers).  Its stage backend here is a plain stand-in written from the definitions with the oracle's
building blocks (oracle.apply_D for exp(h/2 L), numpy for |A|^2 and the kappa rows) — test infrastructure, not a
product fallback.  Two ranks, each holding half of the modes, must reproduce the unsharded oracle."""
import os
import socket

import numpy as np
import pytest

from paper_1901_01895_b200 import sharded, workloads


class OracleShardStages:
    """begin / powers / apply / linear / end of sharded.propagate on numpy arrays, from Eq. (1) and Eq. (6)."""

    def __init__(self, M_total, mode0, N, dt, h, alpha, beta_local, gamma, kappa_rows, chunks=1):
        import torch
        from oracle import oracle
        self.orc = oracle
        self.mode0, self.m, self.N = mode0, len(beta_local), N
        self.hg = h * gamma
        self.kappa_rows = np.asarray(kappa_rows)
        self.E = oracle.linear_table(self.m, N, dt, 0.5 * h, alpha, beta_local)
        self.ranges = sharded.chunk_ranges(N, chunks)
        self.P_all = torch.zeros((chunks, M_total, N // chunks), dtype=torch.float64)

    def begin(self, A):
        self.X = A
        self.Y = np.zeros_like(A)
        self.Z = np.zeros_like(A)
        self.W = np.zeros_like(A)

    def _arg(self, stage, sl):
        return (self.X[:, sl], self.X[:, sl] + 0.5 * self.Y[:, sl], self.X[:, sl] + 0.5 * self.Z[:, sl], self.W[:, sl])[stage]

    def powers(self, stage, c=0):
        t0, n = self.ranges[c]
        u = self._arg(stage, slice(t0, t0 + n))
        self.P_all[c].numpy()[self.mode0:self.mode0 + self.m] = np.abs(u[0::2]) ** 2 + np.abs(u[1::2]) ** 2

    def apply(self, stage, c=0, gain=1.0):
        t0, n = self.ranges[c]
        sl = slice(t0, t0 + n)
        u = self._arg(stage, sl)
        S = self.kappa_rows @ self.P_all[c].numpy()                  # [m][n]
        k = 1j * self.hg * np.repeat(S, 2, axis=0) * u
        if stage == 0:
            self.Y[:, sl] = k
        elif stage == 1:
            self.Z[:, sl] = k
        elif stage == 2:
            self.W[:, sl] = self.X[:, sl] + k
            self.Z[:, sl] = self.X[:, sl] + self.Y[:, sl] / 6 + self.Z[:, sl] / 3 + k / 3
        else:
            self.X[:, sl] = gain * (self.Z[:, sl] + k / 6)

    def linear(self, which):
        for buf in ((self.X, self.Y) if which == 0 else (self.W, self.Z)):
            buf[:] = self.orc.apply_D(buf, self.E)

    def end(self):
        pass


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out, M, N, steps, chunks):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group(backend="gloo", rank=rank, world_size=world)
    try:
        p = workloads.problem(0, M=M, N=N, steps=steps)
        A = p.field() * 30.0                                   # strong enough for the nonlinear term to matter
        mode0, m, beta_l, kappa_rows = sharded.shard_arguments(p.beta, p.kappa, rank, world)
        st = OracleShardStages(p.M, mode0, p.N, p.dt, p.h, p.alpha, beta_l, p.gamma, kappa_rows, chunks=chunks)
        mine = np.ascontiguousarray(A[2 * mode0:2 * (mode0 + m)])
        # chunks > 1: asynchronous gathers, waited for chunk by chunk (the pipelined form the GPU path runs)
        sharded.propagate(st, mine, steps, lambda c: sharded.all_gather_rows(st.P_all[c], mode0, m, dist, async_op=chunks > 1),
                          span=2, gain=1.01)
        out.put((rank, mode0, m, mine))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("chunks", [1, 4])
def test_two_ranks_reproduce_the_unsharded_oracle(chunks):
    import torch.multiprocessing as mp
    from oracle import oracle
    oracle.build()
    M, N, steps = 4, 256, 4
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out, M, N, steps, chunks)) for r in range(2)]
    for pr in procs:
        pr.start()
    res = sorted((out.get(timeout=180) for _ in procs), key=lambda t: t[0])
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    p = workloads.problem(0, M=M, N=N, steps=steps)
    A = p.field() * 30.0
    want = oracle.rk4ip_spans(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 2, 2, 1.01)
    nl = oracle.rk4ip_spans(A, p.dt, p.h, p.alpha, p.beta, 0.0, p.kappa, 2, 2, 1.01)
    assert workloads.rel_l2_per_field(nl, want).min() > 1e-4      # the nonlinear term (and so the gather) matters
    got = np.concatenate([r[3] for r in res], axis=0)
    assert [(r[1], r[2]) for r in res] == [(0, 2), (2, 2)]
    assert workloads.rel_l2_per_field(got, want).max() <= 1e-12


def test_partition():
    assert sharded.mode_range(120, 3, 8) == (45, 15)
    assert sharded.mode_range(6, 0, 1) == (0, 6)
    with pytest.raises(ValueError):
        sharded.mode_range(10, 0, 4)
    with pytest.raises(ValueError):
        sharded.mode_range(8, 2, 2)
    beta = np.arange(12.0).reshape(4, 3)
    kappa = np.arange(16.0).reshape(4, 4)
    mode0, m, b, k = sharded.shard_arguments(beta, kappa, 1, 2)
    assert (mode0, m) == (2, 2) and np.array_equal(b, beta[2:4]) and np.array_equal(k, kappa[2:4, :])


def test_single_process_gather_is_a_no_op():
    import torch
    P = torch.arange(12.0, dtype=torch.float64).reshape(4, 3)
    Q = P.clone()
    assert sharded.all_gather_rows(P, 0, 4, None) is None
    assert torch.equal(P, Q)
    assert sharded.chunk_ranges(256, 4) == [(0, 64), (64, 64), (128, 64), (192, 64)]
    with pytest.raises(ValueError):
        sharded.chunk_ranges(256, 16)


def test_propagate_detaches_the_field_when_a_stage_fails():
    """sharded.propagate calls stages.end() in a finally block: a stage that raises must not leave A attached."""
    from paper_1901_01895_b200 import sharded

    class Failing:
        ranges = [(0, 16)]
        log = []

        def begin(self, A):
            self.log.append("begin")

        def powers(self, stage, c=0):
            self.log.append("powers")

        def apply(self, stage, c=0, gain=1.0):
            raise RuntimeError("apply failed")

        def linear(self, which):
            self.log.append("linear")

        def end(self):
            self.log.append("end")

    st = Failing()
    with pytest.raises(RuntimeError, match="apply failed"):
        sharded.propagate(st, None, 2, lambda c: None)
    assert st.log == ["begin", "powers", "end"]
