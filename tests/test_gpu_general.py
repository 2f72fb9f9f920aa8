"""GPU parity of the GENERAL per-polarisation coupling: mmf_plan_create_general +
mmf_apply_nonlinear / mmf_propagate against the oracle's nonlinear_general / rk4ip_general on the same seeded inputs.
Bit-exact on integers (non-symmetric integer 2M x 2M matrix), <= 1e-10 relative L2 per field after propagation."""
import numpy as np
import pytest

from paper_1901_01895_b200 import workloads

pytestmark = pytest.mark.gpu
TOL_FIELD = 1e-10


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    return torch


@pytest.fixture(scope="module")
def mmf():
    from paper_1901_01895_b200 import binding
    binding.lib()
    return binding


def general_kappa(p, seed=0):
    return p.kappa_general(seed)


@pytest.mark.parametrize("M,N", [(1, 16), (4, 64), (5, 32), (37, 128), (64, 64), (120, 256)])
def test_general_nonlinear_integer_exact(mmf, torch, orc, M, N):
    rng = np.random.default_rng(M * 1000 + N)
    R = 2 * M
    u = (rng.integers(-30, 31, size=(R, N)) + 1j * rng.integers(-30, 31, size=(R, N))).astype(complex)
    k2 = rng.integers(-9, 10, size=(R, R)).astype(float)
    pl = mmf.Plan(M, N, 1.0, 1.0, 0.0, np.zeros((M, 1)), 1.0, k2, general=True)
    U = torch.from_numpy(u).to("cuda:0")
    OUT = torch.empty_like(U)
    pl.apply_nonlinear(U, OUT)
    want = orc.nonlinear_general(u, 1.0, k2)
    assert np.array_equal(OUT.cpu().numpy(), want)
    pl.apply_nonlinear(U, U)                        # exact aliasing goes through the workspace
    assert np.array_equal(U.cpu().numpy(), want)


def test_general_reduces_to_manakov(mmf, torch):
    """kappa2[2a+p][2b+q] = kappa_ab: the general plan must reproduce the Manakov plan (rounding-level difference:
    the sums run over 2M instead of M terms)."""
    p = workloads.problem(3, M=37, N=1 << 13, steps=3)
    A = p.field() * 3.0
    X1 = torch.from_numpy(A).to("cuda:0")
    X2 = X1.clone()
    mmf.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa).propagate(X1, 3)
    mmf.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, np.kron(p.kappa, np.ones((2, 2))), general=True).propagate(X2, 3)
    assert workloads.rel_l2_per_field(X2.cpu().numpy(), X1.cpu().numpy()).max() <= 1e-13


# 2M = 8, 74, 240 (SURVEY/VERDICT), single-pass and three-pass transforms, odd M (the half boundary splits a mode)
CASES = [(0, 4, 12, 50), (0, 2, 9, 5), (2, 37, 13, 4), (3, 120, 13, 3), (3, 120, 14, 2), (4, 7, 18, 3), (1, 6, 16, 10)]


@pytest.mark.parametrize("cfg,M,logn,steps", CASES)
def test_general_propagate_matches_oracle(mmf, torch, orc, cfg, M, logn, steps):
    p = workloads.problem(cfg, M=M, N=1 << logn, steps=steps)
    A = p.field() * 3.0
    k2 = general_kappa(p)
    pl = mmf.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, k2, general=True)
    X = torch.from_numpy(A).to("cuda:0")
    pl.propagate(X, steps)
    torch.cuda.synchronize()
    want = orc.rk4ip_general(A, p.dt, p.h, p.alpha, p.beta, p.gamma, k2, steps)
    err = workloads.rel_l2_per_field(X.cpu().numpy(), want)
    assert workloads.rel_l2_per_field(want, A).min() > 1e-6
    assert err.max() <= TOL_FIELD, (err.max(), err.argmax())


def test_general_composes_and_rejects_split_step(mmf, torch):
    import ctypes
    p = workloads.problem(1, M=3, N=1 << 13, steps=5)
    A = p.field()
    k2 = general_kappa(p)
    pl = mmf.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, k2, general=True)
    X = torch.from_numpy(A).to("cuda:0")
    pl.propagate(X, 5)
    Y = torch.from_numpy(A).to("cuda:0")
    pl.propagate(Y, 2)
    pl.propagate(Y, 3)
    assert np.array_equal(Y.cpu().numpy(), X.cpu().numpy())
    L = mmf.lib()
    assert L.mmf_propagate_ssfm(pl._h, ctypes.c_void_p(X.data_ptr()), 1, None) == mmf.MMF_EINVAL
    assert L.mmf_propagate_ssfm_agrawal(pl._h, ctypes.c_void_p(X.data_ptr()), 1, 2, None) == mmf.MMF_EINVAL
    rc, h = mmf.raw_create(121, 4096, 1.0, 1.0, 0.0, np.zeros((121, 1)), 1, 0.0, np.zeros((242, 242)), general=True)
    assert rc == mmf.MMF_EINVAL


def test_general_cfg4_timed_plan_sampled_samples(mmf, torch, orc):
    """the 240 x 2^22 plan with the general matrix, dispersion off: the step acts sample by sample, the oracle computes
    sampled time samples one by one (two steps, <= 1e-10)."""
    p = workloads.problem(4)
    rng = np.random.default_rng(46)
    idx = np.sort(np.unique(np.concatenate([[0, 7, 8, p.N - 1], rng.integers(0, p.N, size=256)]))[:64])
    small = workloads.problem(4, N=1 << 16).field() * 10.0
    X = torch.from_numpy(small).to("cuda:0").repeat(1, p.N >> 16).contiguous()
    sub = np.ascontiguousarray(small[:, idx % (1 << 16)])
    k2 = general_kappa(p)
    pl = mmf.Plan(p.M, p.N, p.dt, p.h, 0.0, np.zeros_like(p.beta), p.gamma, k2, general=True)
    pl.propagate(X, 2)
    got = X[:, torch.from_numpy(idx).to("cuda:0")].cpu().numpy()
    want = orc.rk4ip_general(sub, p.dt, p.h, 0.0, np.zeros_like(p.beta), p.gamma, k2, 2)
    assert workloads.rel_l2_per_field(want, sub).min() > 1e-3
    assert workloads.rel_l2_per_field(got, want).max() <= TOL_FIELD
