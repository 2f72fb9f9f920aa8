"""Mode groups (section 6): a kappa with few distinct rows runs the grouped contraction of
nl_tma.cuh (G M instead of M M products per sample).  The values must not change: against the oracle (which knows
nothing of groups: it sums the dense matrix) and against the dense CUDA contraction of the same matrix."""
import numpy as np
import pytest

from paper_1901_01895_b200 import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def mmf():
    from paper_1901_01895_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def orc():
    from oracle import oracle
    oracle.build()
    return oracle


def _plan(mmf, p, kappa):
    return mmf.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, kappa)


@pytest.mark.parametrize("M,N", [(10, 64), (36, 128), (120, 256), (55, 32)])
def test_grouped_nonlinear_integer_exact(mmf, torch, orc, M, N):
    """Gaussian-integer field, integer NON-symmetric group matrix: bit-exact against the oracle's dense sum."""
    rng = np.random.default_rng(M * 7 + N)
    p = workloads.problem(3, M=M, N=N)
    _, group_of = p.kappa_grouped()
    G = int(group_of.max()) + 1
    K = rng.integers(-9, 10, size=(G, M)).astype(float)          # distinct ROWS; columns unconstrained
    kap = K[group_of]
    u = rng.integers(-30, 31, size=(2 * M, N)) + 1j * rng.integers(-30, 31, size=(2 * M, N))
    pl = mmf.Plan(M, N, 1.0, 1.0, 0.0, np.zeros((M, 1)), 1.0, kap)
    assert pl.groups() == len({tuple(r) for r in kap})
    U = torch.from_numpy(u.astype(np.complex128)).cuda()
    OUT = torch.empty_like(U)
    pl.apply_nonlinear(U, OUT)
    torch.cuda.synchronize()
    want = orc.nonlinear(u.astype(np.complex128), 1.0, kap)
    assert np.array_equal(OUT.cpu().numpy(), want)


@pytest.mark.parametrize("cfg,M,logn,steps", [(3, 120, 13, 3), (2, 36, 14, 3), (0, 10, 12, 4), (1, 21, 16, 2)])
def test_grouped_propagation_matches_oracle_and_dense_path(mmf, torch, orc, monkeypatch, cfg, M, logn, steps):
    p = workloads.problem(cfg, M=M, N=1 << logn, steps=steps)
    kap, group_of = p.kappa_grouped()
    A = p.field() * 6.0
    want = orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, steps)
    assert workloads.rel_l2_per_field(orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, 0.0, kap, steps), want).min() > 1e-6
    got = {}
    for flag in ("1", "0"):
        monkeypatch.setenv("MMF_GROUPED", flag)
        pl = _plan(mmf, p, kap)
        assert pl.groups() == (int(group_of.max()) + 1 if flag == "1" else 0)
        X = torch.from_numpy(A).cuda()
        pl.propagate(X, steps)
        torch.cuda.synchronize()
        got[flag] = X.cpu().numpy()
        pl.destroy()
    assert workloads.rel_l2_per_field(got["1"], want).max() <= 1e-10
    assert workloads.rel_l2_per_field(got["1"], got["0"]).max() <= 1e-13


def test_grouped_split_steps_and_spans(mmf, torch, orc):
    p = workloads.problem(3, M=28, N=1 << 13, steps=3)
    kap, _ = p.kappa_grouped()
    A = p.field() * 6.0
    pl = _plan(mmf, p, kap)
    assert pl.groups() == 7
    X = torch.from_numpy(A).cuda()
    pl.propagate_ssfm(X, 3)
    torch.cuda.synchronize()
    assert workloads.rel_l2_per_field(X.cpu().numpy(), orc.ssfm_rk4(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, 3)).max() <= 1e-10
    X = torch.from_numpy(A).cuda()
    pl.propagate_ssfm_agrawal(X, 3, niter=2)
    torch.cuda.synchronize()
    assert workloads.rel_l2_per_field(X.cpu().numpy(), orc.ssfm_agrawal(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, 3, niter=2)).max() <= 1e-10
    g = float(np.exp(p.alpha * p.h))
    X = torch.from_numpy(A).cuda()
    pl.propagate_spans(X, 2, 2, g)
    torch.cuda.synchronize()
    assert workloads.rel_l2_per_field(X.cpu().numpy(), orc.rk4ip_spans(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, 2, 2, g)).max() <= 1e-10


def test_dense_kappa_is_not_grouped(mmf, torch):
    p = workloads.problem(2, M=12, N=1 << 12)
    assert _plan(mmf, p, p.kappa).groups() == 0                       # all rows distinct
    ones = np.ones((12, 12))
    assert _plan(mmf, p, ones).groups() == 1                          # one group
    two = np.ones((12, 12)); two[7:] = 2.0
    assert _plan(mmf, p, two).groups() == 2
    many = np.arange(144.0).reshape(12, 12); many[1] = many[0]
    assert _plan(mmf, p, many).groups() == 0                          # 11 distinct rows > M / 2: dense


def test_many_groups_at_120_modes_all_paths(mmf, torch, orc):
    """M = 120 with 32 distinct rows: the largest split-step slots leave no room for the grouped kernel's S rows, so
    those launches contract the dense matrix (mmf_api.cu); every path must still match the oracle."""
    p = workloads.problem(3, M=120, N=1 << 13, steps=2)
    rng = np.random.default_rng(5)
    group_of = np.arange(120) % 32
    K = rng.uniform(0.01, 0.5, size=(32, 120))
    kap = K[group_of]
    A = p.field() * 6.0
    pl = _plan(mmf, p, kap)
    assert pl.groups() == 32
    for name, fn, ref in (("rk4ip", lambda X: pl.propagate(X, 2), lambda: orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, 2)),
                          ("ssfm", lambda X: pl.propagate_ssfm(X, 2), lambda: orc.ssfm_rk4(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, 2)),
                          ("agrawal", lambda X: pl.propagate_ssfm_agrawal(X, 2, niter=3),
                           lambda: orc.ssfm_agrawal(A, p.dt, p.h, p.alpha, p.beta, p.gamma, kap, 2, niter=3))):
        X = torch.from_numpy(A).cuda()
        fn(X)
        torch.cuda.synchronize()
        assert workloads.rel_l2_per_field(X.cpu().numpy(), ref()).max() <= 1e-10, name
