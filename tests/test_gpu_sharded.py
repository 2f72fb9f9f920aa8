"""Row-sharded RK4IP on the GPU: the stage calls mmf_shard_* of the C ABI, driven by
paper_1901_01895_b200/sharded.py, against the (unsharded) CPU oracle.  One GPU is available, so K ranks are K shard
plans in one process, each with its own field rows and its own gathered-power buffer; the "collective" copies the
rows between those buffers (stream-ordered: no kernel ever waits on another)."""
import threading

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _run_shards(p, A, steps, world, span=0, gain=1.0, chunks=1):
    import torch
    from paper_1901_01895_b200 import sharded
    stages, fields, rng = [], [], []
    for r in range(world):
        mode0, m, beta_l, kappa_rows = sharded.shard_arguments(p.beta, p.kappa, r, world)
        stages.append(sharded.CudaShardStages(p.M, mode0, p.N, p.dt, p.h, p.alpha, beta_l, p.gamma, kappa_rows, chunks=chunks))
        fields.append(torch.from_numpy(np.ascontiguousarray(A[2 * mode0:2 * (mode0 + m)])).cuda())
        rng.append((mode0, m))
    bar = threading.Barrier(world)
    errs = []

    def gather(r, c):
        bar.wait()                      # every rank has enqueued its powers kernel (same stream: ordered)
        for j, (m0, m) in enumerate(rng):
            if j != r:
                stages[r].P_all[c, m0:m0 + m].copy_(stages[j].P_all[c, m0:m0 + m])
        bar.wait()                      # nobody overwrites its rows before everybody has copied them

    def rank(r):
        try:
            torch.cuda.set_device(0)
            sharded.propagate(stages[r], fields[r], steps, lambda c: gather(r, c), span=span, gain=gain)
        except Exception as e:          # pragma: no cover
            errs.append(e)
            bar.abort()

    th = [threading.Thread(target=rank, args=(r,)) for r in range(world)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errs, errs
    torch.cuda.synchronize()
    launches = sum(s.plan.launch_count() for s in stages)
    for s in stages:
        s.plan.destroy()
    return np.concatenate([f.cpu().numpy() for f in fields], axis=0), launches


@pytest.mark.parametrize("cfg,M,logn,steps,world,chunks", [(0, 2, 12, 5, 1, 1), (0, 2, 12, 5, 2, 2), (1, 6, 14, 3, 1, 4),
                                                          (1, 6, 14, 3, 2, 1), (1, 6, 14, 3, 3, 8), (4, 4, 16, 2, 4, 2),
                                                          (2, 12, 8, 3, 4, 1), (2, 12, 8, 3, 4, 8)])
def test_sharded_propagation_matches_oracle(cfg, M, logn, steps, world, chunks):
    from oracle import oracle
    from paper_1901_01895_b200 import workloads
    p = workloads.problem(cfg, M=M, N=1 << logn, steps=steps)
    A = p.field() * (8.0 if cfg < 4 else 1.0)
    got, launches = _run_shards(p, A, steps, world, chunks=chunks)
    want = oracle.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, steps)
    err = workloads.rel_l2_per_field(got, want)
    assert err.max() <= 1e-10, err
    lin = oracle.rk4ip(A, p.dt, p.h, p.alpha, p.beta, 0.0, p.kappa, steps)
    assert workloads.rel_l2_per_field(lin, want).max() > 1e-6        # the coupling across shards matters in this case
    assert launches > 0


def test_sharded_spans_gain():
    from oracle import oracle
    from paper_1901_01895_b200 import workloads
    p = workloads.problem(1, M=4, N=1 << 13, steps=4)
    A = p.field() * 8.0
    g = float(np.exp(p.alpha * p.h * 2 / 2))
    got, _ = _run_shards(p, A, 4, 2, span=2, gain=g)
    want = oracle.rk4ip_spans(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 2, 2, g)
    assert workloads.rel_l2_per_field(got, want).max() <= 1e-10


def test_powers_integer_exact_and_offsets():
    """mmf_shard_powers on Gaussian integers: P_all rows mode0.. bit-exact, the other rows untouched."""
    import torch
    from paper_1901_01895_b200 import sharded, workloads
    p = workloads.problem(0, M=6, N=1 << 12, steps=1)
    rng = np.random.default_rng(7)
    A = (rng.integers(-50, 50, size=(12, p.N)) + 1j * rng.integers(-50, 50, size=(12, p.N))).astype(np.complex128)
    mode0, m, beta_l, kappa_rows = sharded.shard_arguments(p.beta, p.kappa, 1, 3)
    st = sharded.CudaShardStages(p.M, mode0, p.N, p.dt, p.h, p.alpha, beta_l, p.gamma, kappa_rows)
    X = torch.from_numpy(np.ascontiguousarray(A[2 * mode0:2 * (mode0 + m)])).cuda()
    st.P_all.fill_(-1.0)
    st.begin(X)
    st.powers(sharded.SH_PLAIN)
    st.end()
    P = st.P_all[0].cpu().numpy()
    sq = A.real ** 2 + A.imag ** 2                      # exact in fp64 for these integers
    want = sq[0::2] + sq[1::2]
    assert np.array_equal(P[mode0:mode0 + m], want[mode0:mode0 + m])
    assert np.all(P[:mode0] == -1.0) and np.all(P[mode0 + m:] == -1.0)
    st.plan.destroy()


def test_shard_plan_rejects_the_unsharded_calls():
    import torch
    from paper_1901_01895_b200 import binding, sharded, workloads
    p = workloads.problem(0, M=4, N=1 << 12, steps=1)
    mode0, m, beta_l, kappa_rows = sharded.shard_arguments(p.beta, p.kappa, 0, 2)
    st = sharded.CudaShardStages(p.M, mode0, p.N, p.dt, p.h, p.alpha, beta_l, p.gamma, kappa_rows)
    X = torch.zeros((2 * m, p.N), dtype=torch.complex128, device="cuda")
    with pytest.raises(binding.MmfError):
        st.plan.propagate(X, 1)
    with pytest.raises(binding.MmfError):
        st.powers(0)                      # no field attached
    rc, _ = binding.raw_create(2, 4096, 1.0, 1.0, 0.0, np.zeros((2, 4)), 4, 1.0, np.ones((2, 2)))
    assert rc == binding.MMF_OK
    st.plan.destroy()
