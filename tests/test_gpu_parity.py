"""GPU parity tests: the CUDA path (through the C ABI of include/mmf.h) against the CPU oracle, element by element on
the same seeded inputs.  Bars: bit-exact for integer / index work; relative L2 <= 1e-10 per field for propagated
fields (BASELINE.json north_star); tighter, arithmetic-derived bounds for single operators.
"""
import numpy as np
import pytest

from paper_1901_01895_b200 import workloads

pytestmark = pytest.mark.gpu

TOL_FIELD = 1e-10          # north_star: relative L2 per field after the stated number of steps
TOL_OP = 2e-14             # one transform pair / one operator: ~ log2(N) * eps, generous


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    return torch


@pytest.fixture(scope="module")
def mmf():
    from paper_1901_01895_b200 import binding
    binding.lib()           # fail loudly if the CUDA library is missing
    return binding


def to_dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def plan_for(mmf, p, **over):
    kw = dict(M=p.M, N=p.N, dt=p.dt, h=p.h, alpha=p.alpha, beta=p.beta, gamma=p.gamma, kappa=p.kappa)
    kw.update(over)
    return mmf.Plan(**kw)


def rand_c(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


# ------------------------------------------------------------------------------------------ index permutation (P10 i)
@pytest.mark.parametrize("logn", [4, 5, 9, 12, 13, 16, 18, 22])
def test_slot_map_is_a_permutation(mmf, torch, logn):
    N = 1 << logn
    pl = mmf.Plan(1, N, 1.0, 1.0, 0.0, np.zeros((1, 1)), 0.0, np.ones((1, 1)))
    idx = pl.debug_freq_index()
    assert idx.min() == 0 and idx.max() == N - 1
    assert np.array_equal(np.sort(idx), np.arange(N))


# ----------------------------------------------------------------------------------------------- forward transform
@pytest.mark.parametrize("logn", [4, 6, 7, 11, 12, 13, 14, 16])
def test_forward_transform_matches_oracle(mmf, torch, orc, logn):
    N, M = 1 << logn, 2
    rng = np.random.default_rng(logn)
    x = rand_c(rng, 2 * M, N)
    pl = mmf.Plan(M, N, 1.0, 1.0, 0.0, np.zeros((M, 1)), 0.0, np.eye(M))
    X = to_dev(torch, x)
    S = torch.empty_like(X)
    pl.debug_forward(X, S)
    got = S.cpu().numpy()
    for r in range(2 * M):
        want = orc.fft(x[r], +1)
        assert workloads.rel_l2_per_field(got[r], want) <= TOL_OP


@pytest.mark.parametrize("logn", [4, 8, 12, 14])
def test_forward_transform_integer_exact(mmf, torch, orc, logn):
    """Gaussian integers on every (N/4)-th sample: only the twiddles 1, i, -1, -i meet non-zero data, all sums are
    exact in fp64, so CUDA and oracle must agree BIT FOR BIT (P10 iii)."""
    N, M = 1 << logn, 1
    rng = np.random.default_rng(100 + logn)
    x = np.zeros((2, N), dtype=complex)
    x[:, :: N // 4] = rng.integers(-1000, 1000, size=(2, 4)) + 1j * rng.integers(-1000, 1000, size=(2, 4))
    pl = mmf.Plan(M, N, 1.0, 1.0, 0.0, np.zeros((M, 1)), 0.0, np.eye(M))
    X = to_dev(torch, x)
    S = torch.empty_like(X)
    pl.debug_forward(X, S)
    got = S.cpu().numpy()
    for r in range(2):
        assert np.array_equal(got[r], orc.fft(x[r], +1))


# ------------------------------------------------------------------------------------------------ linear operator D
@pytest.mark.parametrize("cfg,M,logn", [(0, 2, 12), (1, 3, 13), (1, 2, 16), (2, 3, 14), (3, 5, 18), (4, 2, 15), (4, 1, 4),
                                        (4, 1, 22), (4, 1, 23)] +
                         # every transform length the plan accepts (each (N1, N2) split is its own instantiation)
                         [(4, 1 + (logn & 1), logn) for logn in range(5, 25) if logn not in (12, 13, 14, 15, 16, 18, 22, 23)])
def test_linear_operator_matches_oracle(mmf, torch, orc, cfg, M, logn):
    p = workloads.problem(cfg, M=M, N=1 << logn)
    A = p.field()
    pl = plan_for(mmf, p)
    X = to_dev(torch, A)
    pl.apply_linear(X)
    got = X.cpu().numpy()
    E = orc.linear_table(p.M, p.N, p.dt, p.h / 2, p.alpha, p.beta, nthreads=orc.default_threads())
    want = orc.apply_D(A, E, nthreads=orc.default_threads())
    err = workloads.rel_l2_per_field(got, want)
    assert err.max() <= 5e-14, err


def test_linear_operator_white_input_all_bins(mmf, torch, orc):
    """White (all-bin) input exercises every entry of the exp(h/2 L) table including the Nyquist bin."""
    M, N = 2, 1 << 13
    p = workloads.problem(4, M=M, N=N)
    A = rand_c(np.random.default_rng(8), 2 * M, N)
    pl = plan_for(mmf, p)
    X = to_dev(torch, A)
    pl.apply_linear(X)
    E = orc.linear_table(M, N, p.dt, p.h / 2, p.alpha, p.beta)
    want = orc.apply_D(A, E)
    assert workloads.rel_l2_per_field(X.cpu().numpy(), want).max() <= 5e-14


# --------------------------------------------------------------------------------------------- nonlinear operator
@pytest.mark.parametrize("M,N", [(1, 16), (5, 64), (8, 64), (24, 32), (37, 128), (120, 256), (121, 16), (130, 32)])
def test_nonlinear_operator_integer_exact(mmf, torch, orc, M, N):
    """P10 ii: Gaussian-integer field, integer NON-symmetric kappa, h*gamma = 1: bit-exact against the oracle."""
    rng = np.random.default_rng(M * 1000 + N)
    u = rng.integers(-30, 31, size=(2 * M, N)) + 1j * rng.integers(-30, 31, size=(2 * M, N))
    kap = rng.integers(-9, 10, size=(M, M)).astype(float)
    pl = mmf.Plan(M, N, 1.0, 1.0, 0.0, np.zeros((M, 1)), 1.0, kap)
    U = to_dev(torch, u.astype(complex))
    OUT = torch.empty_like(U)
    pl.apply_nonlinear(U, OUT)
    want = orc.nonlinear(u.astype(complex), 1.0, kap)
    assert np.array_equal(OUT.cpu().numpy(), want)
    pl.apply_nonlinear(U, U)                        # exact aliasing is allowed
    assert np.array_equal(U.cpu().numpy(), want)


@pytest.mark.parametrize("cfg,M,logn", [(0, 2, 12), (2, 36, 10), (3, 120, 9)])
def test_nonlinear_operator_matches_oracle(mmf, torch, orc, cfg, M, logn):
    p = workloads.problem(cfg, M=M, N=1 << logn)
    A = p.field() * 30.0
    pl = plan_for(mmf, p)
    U = to_dev(torch, A)
    OUT = torch.empty_like(U)
    pl.apply_nonlinear(U, OUT)
    want = orc.nonlinear(A, p.h * p.gamma, p.kappa, nthreads=orc.default_threads())
    assert workloads.rel_l2_per_field(OUT.cpu().numpy(), want).max() <= 1e-14


# ----------------------------------------------------------------------------------------------- the RK4IP step
# (config, M, log2 N, steps): shrunken versions of the five configs of BASELINE.json that the oracle finishes in
# seconds, spanning single-pass (N <= 4096) and three-pass transforms, ragged mode counts and several time tiles.
CASES = [
    (0, 2, 12, 100),      # config 0 at full size and step count
    (1, 6, 13, 40),
    (1, 6, 16, 12),       # config 1 at full size, shortened
    (1, 6, 16, 1000),     # config 1 at full size and step count
    (2, 36, 14, 8),
    (3, 120, 13, 4),
    (4, 120, 14, 3),
    (4, 7, 18, 3),        # config-4 physics at the 2^18 transform size, odd mode count
    (3, 124, 13, 2),      # more than 120 modes: the DFMA nonlinear kernels and the four-buffer plan
    (4, 1, 23, 1),        # N = 2^23: N1 = 2^12, one-column tiles (W = 1) inside 16-column blocks
    (4, 2, 17, 2), (4, 1, 19, 2), (4, 2, 20, 1), (4, 1, 21, 1), (4, 1, 24, 1),   # the remaining (N1, N2) splits
    (0, 1, 5, 3), (0, 2, 8, 3), (0, 1, 9, 3), (0, 2, 10, 3),                      # short single-pass transforms
]


@pytest.mark.parametrize("cfg,M,logn,steps", CASES)
def test_propagate_matches_oracle(mmf, torch, orc, cfg, M, logn, steps):
    p = workloads.problem(cfg, M=M, N=1 << logn, steps=steps)
    A = p.field()
    pl = plan_for(mmf, p)
    X = to_dev(torch, A)
    pl.propagate(X, steps)
    torch.cuda.synchronize()
    got = X.cpu().numpy()
    want = orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, steps)
    err = workloads.rel_l2_per_field(got, want)
    assert workloads.rel_l2_per_field(want, A).min() > 1e-6          # the propagation did something
    assert err.max() <= TOL_FIELD, (err.max(), err.argmax())


def test_propagate_composes_and_zero_steps(mmf, torch, orc):
    """mmf_propagate(n1) then (n2) == (n1+n2) (checks the fused next-step bracket); nsteps = 0 is a no-op."""
    p = workloads.problem(1, M=3, N=1 << 13, steps=5)
    A = p.field()
    pl = plan_for(mmf, p)
    X = to_dev(torch, A)
    pl.propagate(X, 0)
    assert np.array_equal(X.cpu().numpy(), A)
    pl.propagate(X, 5)
    Y = to_dev(torch, A)
    pl.propagate(Y, 2)
    pl.propagate(Y, 3)
    assert workloads.rel_l2_per_field(Y.cpu().numpy(), X.cpu().numpy()).max() <= 1e-14


def test_zero_field_stays_zero(mmf, torch):
    p = workloads.problem(0, N=1 << 12, steps=3)
    A = p.field()
    A[2] = 0
    pl = plan_for(mmf, p)
    X = to_dev(torch, A)
    pl.propagate(X, 3)
    out = X.cpu().numpy()
    assert np.all(out[2] == 0) and np.any(out[3] != 0)


def test_propagate_host_entry_point(mmf, torch, orc):
    p = workloads.problem(0, N=1 << 12, steps=4)
    A = p.field()
    pl = plan_for(mmf, p)
    H = torch.from_numpy(A.copy()).pin_memory()
    scratch = torch.empty((2 * p.M, p.N), dtype=torch.complex128, device="cuda:0")
    pl.propagate_host(H, scratch, 4)
    want = orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 4)
    assert workloads.rel_l2_per_field(H.numpy(), want).max() <= TOL_FIELD
    assert pl.launch_count() > 0


def test_error_paths_on_device(mmf, torch):
    p = workloads.problem(0, N=1 << 12)
    pl = plan_for(mmf, p)
    X = torch.zeros((2 * p.M, p.N), dtype=torch.complex128, device="cuda:0")
    import ctypes
    L = mmf.lib()
    assert L.mmf_propagate(pl._h, ctypes.c_void_p(X.data_ptr()), -1, None) == mmf.MMF_EINVAL
    assert L.mmf_propagate(pl._h, None, 1, None) == mmf.MMF_EINVAL
    assert L.mmf_propagate(pl._h, ctypes.c_void_p(X.data_ptr() + 8), 1, None) == mmf.MMF_EINVAL
    assert L.mmf_plan_set_workspace(pl._h, ctypes.c_void_p(pl._ws_ptr), 16, None) == mmf.MMF_EINVAL


# ------------------------------------------------------------------------------------------ parameter edge cases
@pytest.mark.parametrize("K,logn", [(1, 12), (2, 13), (6, 13), (8, 12)])
def test_linear_operator_any_number_of_beta_terms(mmf, torch, orc, K, logn):
    """K Taylor coefficients beta_0..beta_{K-1}, all non-zero, per mode different (Eq. 1, reading R2)."""
    M, N, dt, h, alpha = 3, 1 << logn, 0.5, 40.0, 3e-4
    rng = np.random.default_rng(K * 100 + logn)
    beta = rng.uniform(-1, 1, size=(M, K)) * (0.02 / (np.arange(K) + 1.0) ** 3)[None, :]
    X = rand_c(rng, 2 * M, N)
    X[:, N // 2] = 0
    A = np.fft.ifft(X, axis=1)
    pl = mmf.Plan(M, N, dt, h, alpha, beta, 0.0, np.eye(M))
    D = to_dev(torch, A)
    pl.apply_linear(D)
    E = orc.linear_table(M, N, dt, h / 2, alpha, beta)
    want = orc.apply_D(A, E)
    assert workloads.rel_l2_per_field(D.cpu().numpy(), want).max() <= 5e-14


def test_propagate_non_symmetric_kappa_no_loss_single_sample_tile(mmf, torch, orc):
    """kappa not symmetric, alpha = 0, K = 3, M = 5 (ragged mode groups), N = 16 (the smallest transform)."""
    M, N, dt, h, steps = 5, 16, 1.0, 0.5, 6
    rng = np.random.default_rng(2024)
    A = rand_c(rng, 2 * M, N) * 0.5
    beta = rng.uniform(-0.05, 0.05, size=(M, 3))
    kappa = rng.uniform(0.1, 1.0, size=(M, M))
    pl = mmf.Plan(M, N, dt, h, 0.0, beta, 0.1, kappa)
    X = to_dev(torch, A)
    pl.propagate(X, steps)
    want = orc.rk4ip(A, dt, h, 0.0, beta, 0.1, kappa, steps)
    assert workloads.rel_l2_per_field(want, A).min() > 1e-3
    assert workloads.rel_l2_per_field(X.cpu().numpy(), want).max() <= TOL_FIELD


# ------------------------------------------------------------------------ spans with lumped amplifiers
@pytest.mark.parametrize("cfg,M,logn,nspans,k,general", [(0, 2, 12, 3, 4, False), (1, 6, 14, 2, 3, False),
                                                          (3, 120, 13, 2, 2, False), (3, 122, 13, 2, 2, False),
                                                          (2, 5, 13, 2, 3, True), (1, 3, 16, 1, 40, False)])
def test_spans_match_oracle(mmf, torch, orc, cfg, M, logn, nspans, k, general):
    """mmf_propagate_spans: the amplifier gain rides on the last kernel of every span (graph-replayed bodies in
    between for the small cases); against the oracle's rk4ip_spans."""
    import math
    p = workloads.problem(cfg, M=M, N=1 << logn)
    A = p.field() * 2.0
    kap = p.kappa_general() if general else p.kappa
    gain = math.exp(p.alpha * p.h * k / 2) * 1.7          # more than the loss: the nonlinearity grows span by span
    pl = mmf.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, general=general)
    X = to_dev(torch, A)
    pl.propagate_spans(X, nspans, k, gain)
    want = orc.rk4ip_spans(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, nspans, k, gain, general=general)
    err = workloads.rel_l2_per_field(X.cpu().numpy(), want)
    assert err.max() <= TOL_FIELD, (err.max(), err.argmax())
    nogain = orc.rk4ip_spans(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, nspans, k, 1.0, general=general)
    assert workloads.rel_l2_per_field(want, nogain).min() > 0.1


def test_graph_replay_is_bit_identical_to_direct_launches(mmf, torch, monkeypatch):
    """small problems replay their step body from a CUDA graph; with per-launch timing on they launch directly:
    both must give the same bits, for step counts that mix 16-step graphs, 1-step graphs and the direct tail.
    (The kernel-per-stage plan is selected explicitly: at this size mmf_propagate would run as one cluster kernel.)"""
    monkeypatch.setenv("MMF_SMALL_CLUSTER", "0")
    p = workloads.problem(0, N=1 << 12)
    A = p.field()
    pl = plan_for(mmf, p)
    for steps in (1, 2, 3, 18, 37):
        X = to_dev(torch, A)
        n0 = pl.launch_count()
        pl.propagate(X, steps)
        n_graph = pl.launch_count() - n0
        Y = to_dev(torch, A)
        pl.set_timing(True)
        n0 = pl.launch_count()
        pl.propagate(Y, steps)
        n_direct = pl.launch_count() - n0
        pl.set_timing(False)
        assert np.array_equal(X.cpu().numpy(), Y.cpu().numpy()), steps
        assert n_graph == n_direct == 1 + 4 * steps


def test_propagate_host_batch(mmf, torch, orc):
    """five host fields (a launch-power sweep) through two device buffers with overlapped copies; every field must
    come back as the oracle propagates it."""
    p = workloads.problem(1, M=3, N=1 << 14, steps=4)
    A = p.field()
    scales = [0.5, 1.0, 1.5, 2.0, 2.5]
    hosts = [torch.from_numpy(A * s).pin_memory() for s in scales]
    pl = plan_for(mmf, p)
    d0 = torch.empty((2 * p.M, p.N), dtype=torch.complex128, device="cuda:0")
    d1 = torch.empty_like(d0)
    pl.propagate_host_batch(hosts, d0, d1, 4)
    for H, s in zip(hosts, scales):
        want = orc.rk4ip(A * s, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 4)
        assert workloads.rel_l2_per_field(H.numpy(), want).max() <= TOL_FIELD
    pl.propagate_host_batch(hosts[:1], d0, None, 0)                       # one field, zero steps: a round trip


# ------------------------------------------------------------------------------- whole-propagation cluster kernel
@pytest.mark.parametrize("M,steps", [(1, 6), (2, 9), (3, 5), (4, 4)])
def test_small_cluster_kernel_matches_oracle_and_the_launch_by_launch_plan(mmf, torch, orc, monkeypatch, M, steps):
    """N = 4096, M <= 4: mmf_propagate runs as ONE cluster kernel (small_cluster.cuh: the field in distributed shared
    memory, D and N alternating with cluster barriers).  Against the oracle, and against the kernel-per-stage plan
    (MMF_SMALL_CLUSTER=0), which must give the same field to rounding."""
    p = workloads.problem(0, M=M, N=1 << 12, steps=steps)
    A = p.field() * 20.0
    want = orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, steps)
    assert workloads.rel_l2_per_field(orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, 0.0, p.kappa, steps), want).min() > 1e-4
    got = {}
    for mode in ("1", "0"):
        monkeypatch.setenv("MMF_SMALL_CLUSTER", mode)
        pl = plan_for(mmf, p)
        X = to_dev(torch, A)
        n0 = pl.launch_count()
        pl.propagate(X, steps)
        torch.cuda.synchronize()
        got[mode] = (X.cpu().numpy(), pl.launch_count() - n0)
        pl.destroy()
    assert got["1"][1] == 1 and got["0"][1] > 1                 # one launch for the whole call
    for mode in ("1", "0"):
        assert workloads.rel_l2_per_field(got[mode][0], want).max() <= 1e-10
    assert workloads.rel_l2_per_field(got["1"][0], got["0"][0]).max() <= 1e-13


def test_small_cluster_kernel_spans_and_composition(mmf, torch, orc):
    p = workloads.problem(0, M=2, N=1 << 12, steps=6)
    A = p.field() * 20.0
    g = float(np.exp(p.alpha * p.h * 3 / 2))
    pl = plan_for(mmf, p)
    X = to_dev(torch, A)
    pl.propagate_spans(X, 2, 3, g)
    torch.cuda.synchronize()
    want = orc.rk4ip_spans(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 2, 3, g)
    assert workloads.rel_l2_per_field(X.cpu().numpy(), want).max() <= 1e-10
    X1, X2 = to_dev(torch, A), to_dev(torch, A)
    pl.propagate(X1, 6)
    pl.propagate(X2, 2)
    pl.propagate(X2, 4)
    torch.cuda.synchronize()
    assert torch.equal(X1, X2)                                   # n1 + n2 steps == n1 then n2, bit for bit


# ------------------------------------------------------------------------------------ several live plans at once
def test_two_live_plans_sharing_a_kernel_instantiation_interleave(mmf, torch, orc):
    """The opt-in shared-memory limit is a property of (kernel, device), not of a plan.  Two live plans whose launches
    go through the same kernel instantiation with DIFFERENT dynamic shared-memory sizes (M = 8 and M = 7 share one
    k_nlt bucket; two general plans with different M share k_nlg; two M > 120 plans share k_nl) must keep working when
    their calls alternate: the library may only ever raise that limit."""
    def run(cases, **kw):
        plans, fields, wants = [], [], []
        for cfg, M, scale in cases:
            p = workloads.problem(cfg, M=M, N=1 << 13, steps=2)
            A = p.field() * scale
            kap = p.kappa
            if kw.get("general"):
                kap = p.kappa_general(M)
                wants.append(orc.rk4ip_general(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, 4))
            else:
                wants.append(orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, 4))
            plans.append(mmf.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, **kw))
            fields.append(to_dev(torch, A))
        for _ in range(2):                      # larger first, then smaller, then larger again ...
            for pl, X in zip(plans, fields):
                pl.propagate(X, 2)
        torch.cuda.synchronize()
        for X, want in zip(fields, wants):
            assert np.isfinite(want).all()
            assert workloads.rel_l2_per_field(X.cpu().numpy(), want).max() <= TOL_FIELD
        for pl in plans:
            pl.destroy()
    run(((1, 8, 10.0), (1, 7, 10.0)))
    run(((3, 124, 1.0), (3, 122, 1.0)))
    run(((1, 9, 3.0), (1, 5, 3.0)), general=True)
