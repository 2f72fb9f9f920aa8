"""mmf_apply_nonlinear_static — the one entry point of the library that allocates no device memory — against the
plan-based mmf_apply_nonlinear.

Why the entry point exists: some users of this library cannot call cudaMalloc.  A simulator that reserved all of HBM
for its own pool when it started, a framework whose caching allocator has to account for every device byte, and a
latency-critical loop that must not hit the device-wide synchronisation hidden in cudaMalloc / cudaFree can neither
create a plan (that allocates the plan's tables) nor provide a workspace.  For them the nonlinear operator of Eq. (1)
 is offered in the two-kernel form of the paper's Listing 1 with its one intermediate, the real [M][N]
matrix of mode powers, held in a fixed 4 MiB `static __device__` array inside the library.

What is checked here, on the GPU:
  * two calls in a row (different data, the second one SMALLER so that stale powers of the first call sit right behind
    the part of the array it uses; then the first input again) give what the plan-based path gives, within the
    tolerance the other operator tests use (relative L2 per field <= 1e-14; bit for bit on integer data);
  * the calls allocate nothing: torch's allocator statistics and the driver's free-memory figure do not move across a
    call once the first call's set-up is done;
  * a problem beyond the array is refused with MMF_ETOOBIG and a message that says so, the output left untouched.
The file sorts last on purpose (`pytest --collect-only`): under `pytest -x` a failure here hides no other test.  It
passes alone in a fresh process (its first call then does the set-up) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

from paper_1901_01895_b200 import workloads

pytestmark = pytest.mark.gpu

TOL_NL = 1e-14   # tests/test_gpu_parity.py::test_nonlinear_operator_matches_oracle uses the same bound


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "this test needs the B200"
    return torch


@pytest.fixture(scope="module")
def mmf():
    from paper_1901_01895_b200 import binding
    binding.lib()           # fail loudly if the CUDA library is missing
    return binding


def existing_path(mmf, torch, p, A):
    """h N(A) A through a plan: mmf_plan_create + workspace + mmf_apply_nonlinear (the fused tensor-path kernel)."""
    pl = mmf.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa)
    U = torch.from_numpy(A).to("cuda:0")
    OUT = torch.empty_like(U)
    pl.apply_nonlinear(U, OUT)
    torch.cuda.synchronize()
    out = OUT.cpu().numpy()
    pl.destroy()
    return out


def test_static_scratch_entry_point_matches_plan_path_on_two_calls_in_a_row(mmf, torch):
    # first call: 120 modes x 4096 samples = 491 520 powers, 94 % of the array, 128 time tiles, kappa of config 3;
    # second call: 7 modes x 1000 samples (a ragged last tile, N not a power of two is fine: no transform involved)
    p1 = workloads.problem(3, M=120, N=4096)
    p2 = workloads.problem(1, M=7, N=4096)
    A1 = p1.field() * 30.0
    A2 = np.ascontiguousarray((p2.field() * 30.0)[:, :1000])
    want1 = existing_path(mmf, torch, p1, A1)
    want2 = existing_path(mmf, torch, p2, np.ascontiguousarray(p2.field() * 30.0))[:, :1000]   # N acts sample by sample

    # the caller's memory: everything the entry point touches besides its own static array
    k1 = torch.from_numpy(np.ascontiguousarray(p1.kappa)).to("cuda:0")
    k2 = torch.from_numpy(np.ascontiguousarray(p2.kappa)).to("cuda:0")
    U1, U2 = torch.from_numpy(A1).to("cuda:0"), torch.from_numpy(A2).to("cuda:0")
    O1, O2 = torch.empty_like(U1), torch.empty_like(U2)
    torch.cuda.synchronize()

    mmf.apply_nonlinear_static(k1, U1, O1, p1.h, p1.gamma)        # first call on this device: does the set-up
    mmf.apply_nonlinear_static(k2, U2, O2, p2.h, p2.gamma)        # second call, right behind it in the same stream
    torch.cuda.synchronize()
    assert workloads.rel_l2_per_field(O1.cpu().numpy(), want1).max() <= TOL_NL
    assert workloads.rel_l2_per_field(O2.cpu().numpy(), want2).max() <= TOL_NL

    # a third and fourth call: no allocation anywhere (torch's pool and the driver agree), same results again,
    # and OUT may be U itself
    O1.zero_()                 # outside the bracket: in a fresh process torch loads its fill kernel here, which takes memory
    torch.cuda.synchronize()
    before_torch = (torch.cuda.memory_allocated(), torch.cuda.memory_reserved())
    free_before, _ = torch.cuda.mem_get_info()
    mmf.apply_nonlinear_static(k1, U1, O1, p1.h, p1.gamma)
    mmf.apply_nonlinear_static(k2, U2, U2, p2.h, p2.gamma)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert (torch.cuda.memory_allocated(), torch.cuda.memory_reserved()) == before_torch
    assert free_after == free_before, (free_before, free_after)
    assert workloads.rel_l2_per_field(O1.cpu().numpy(), want1).max() <= TOL_NL
    assert workloads.rel_l2_per_field(U2.cpu().numpy(), want2).max() <= TOL_NL


def test_static_scratch_entry_point_is_exact_on_integers(mmf, torch):
    """Gaussian-integer field, integer non-symmetric kappa, h gamma = 1: every product and sum is exact in fp64, so the
    two paths must agree bit for bit whatever their summation order — twice in a row, with different sizes."""
    for M, N in ((37, 128), (5, 77)):
        rng = np.random.default_rng(M * 1000 + N)
        u = (rng.integers(-30, 31, size=(2 * M, N)) + 1j * rng.integers(-30, 31, size=(2 * M, N))).astype(complex)
        kap = rng.integers(-9, 10, size=(M, M)).astype(float)
        U = torch.from_numpy(u).to("cuda:0")
        OUT = torch.empty_like(U)
        mmf.apply_nonlinear_static(torch.from_numpy(kap).to("cuda:0"), U, OUT, 1.0, 1.0)
        if N >= 16 and (N & (N - 1)) == 0:       # plans want a power-of-two N
            pl = mmf.Plan(M, N, 1.0, 1.0, 0.0, np.zeros((M, 1)), 1.0, kap)
            REF = torch.empty_like(U)
            pl.apply_nonlinear(U, REF)
            want = REF.cpu().numpy()
            pl.destroy()
        else:                                    # written out: i S_a u with S_a = sum_b kappa_ab (|u_bx|^2 + |u_by|^2)
            P = (np.abs(u.real) ** 2 + np.abs(u.imag) ** 2).reshape(M, 2, N).sum(axis=1)
            want = 1j * np.repeat(kap @ P, 2, axis=0) * u
        assert np.array_equal(OUT.cpu().numpy(), want)


def test_static_scratch_entry_point_refuses_what_does_not_fit(mmf, torch):
    L = mmf.lib()
    vp = ctypes.c_void_p
    M, N = 129, 4096                              # 528 384 powers > 524 288
    assert M * N * 8 > mmf.STATIC_SCRATCH_BYTES
    kap = torch.zeros(M, M, dtype=torch.float64, device="cuda:0")
    U = torch.ones(2 * M, N, dtype=torch.complex128, device="cuda:0")
    OUT = torch.full_like(U, 7.0)
    rc = L.mmf_apply_nonlinear_static(M, N, 1.0, 1.0, vp(kap.data_ptr()), vp(U.data_ptr()), vp(OUT.data_ptr()), None)
    assert rc == mmf.MMF_ETOOBIG
    assert b"static scratch" in L.mmf_status_string(rc)
    with pytest.raises(mmf.MmfError, match="static scratch"):
        mmf.apply_nonlinear_static(kap, U, OUT, 1.0, 1.0)
    torch.cuda.synchronize()
    assert bool((OUT == 7.0).all())               # nothing was launched
    # the largest problem that does fit is accepted: 128 x 4096 = 524 288 powers exactly
    rc = L.mmf_apply_nonlinear_static(128, N, 1.0, 1.0, vp(kap.data_ptr()), vp(U.data_ptr()), vp(OUT.data_ptr()), None)
    assert rc == mmf.MMF_OK
    torch.cuda.synchronize()
    assert bool((OUT[:256] == 0.0).all()) and bool((OUT[256:] == 7.0).all())      # kappa = 0 -> N = 0; rows beyond 2M untouched
    # plain argument errors stay MMF_EINVAL
    for bad in ((0, N, 1.0), (M, 0, 1.0), (2, 16, float("nan"))):
        assert L.mmf_apply_nonlinear_static(bad[0], bad[1], bad[2], 1.0, vp(kap.data_ptr()), vp(U.data_ptr()),
                                            vp(OUT.data_ptr()), None) == mmf.MMF_EINVAL
    assert L.mmf_apply_nonlinear_static(2, 16, 1.0, 1.0, None, vp(U.data_ptr()), vp(OUT.data_ptr()), None) == mmf.MMF_EINVAL
