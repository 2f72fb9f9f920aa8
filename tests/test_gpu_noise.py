"""Noise loading on the GPU (mmf_add_noise, reading R18) against the CPU oracle: the generator's 32-bit
words bit for bit, the mode powers and the noisy field within the stated tolerances, the edge cases."""
import ctypes

import numpy as np
import pytest

from paper_1901_01895_b200 import workloads

pytestmark = pytest.mark.gpu

TOL_NOISY_FIELD = 1e-13     # relative L2 per field of A + noise (log / sqrt / sincos differ in the last bits)
TOL_NOISE_ALONE = 1e-11     # relative L2 per field of (A + noise) - A: two digits go in the subtraction at 20 dB
TOL_POWER = 1e-13           # mode powers: a sum of N positive terms in a different (fixed) order


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


@pytest.mark.parametrize("seed,row,t0,count", [(0, 0, 0, 1000), (2024, 7, 12345, 4096), ((1 << 63) + 5, 479, (1 << 32) - 100, 300)])
def test_generator_words_bit_exact(mmf, torch, orc, seed, row, t0, count):
    got = mmf.noise_words(seed, row, t0, count).cpu().numpy().view(np.uint32)
    for i in list(range(0, count, max(1, count // 97))) + [count - 1]:
        t = t0 + i
        want = orc.philox4x32_10([t & 0xFFFFFFFF, t >> 32, row, 0], [seed & 0xFFFFFFFF, seed >> 32])
        assert np.array_equal(got[i], want), (i, got[i], want)
    kat = mmf.noise_words(0, 0, 0, 1).cpu().numpy().view(np.uint32)[0]       # the published all-zero vector
    assert [int(x) for x in kat] == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]


@pytest.mark.parametrize("cfg,M,N,osnr_db,nch", [(0, 2, 4096, 20.0, 60), (1, 6, 1 << 16, 20.0, 60), (3, 120, 1 << 13, 13.5, 1),
                                                  (4, 7, 100003, 25.0, 3), (0, 1, 1, 20.0, 1), (1, 3, 777, 0.0, 2)])
def test_add_noise_matches_oracle(mmf, torch, orc, cfg, M, N, osnr_db, nch):
    p = workloads.problem(cfg, M=M, N=1 << max(4, int(N - 1).bit_length()))
    A = np.ascontiguousarray(p.field()[:, :N])          # ragged N: the operation needs no power of two
    dt, ref_bw, seed = 0.0625, 0.0125, 31337 + M         # ps and THz: 12.5 GHz reference bandwidth
    want, want_P = orc.add_noise(A, dt, osnr_db, ref_bw, nch, seed)
    X = torch.from_numpy(A).to("cuda:0")
    P = mmf.add_noise(X, dt, osnr_db, ref_bw, nch, seed)
    torch.cuda.synchronize()
    got = X.cpu().numpy()
    assert np.allclose(P.cpu().numpy(), want_P, rtol=TOL_POWER, atol=0)
    assert workloads.rel_l2_per_field(got, want).max() <= TOL_NOISY_FIELD
    assert workloads.rel_l2_per_field(got - A, want - A).max() <= TOL_NOISE_ALONE
    assert workloads.rel_l2_per_field(got, A).min() > 1e-4            # noise was really added


def test_add_noise_edge_cases(mmf, torch, orc):
    M, N = 3, 2048
    p = workloads.problem(1, M=M, N=N)
    A = p.field()
    A[2:4] = 0.0                                                      # a dark mode gets no noise
    X = torch.from_numpy(A).to("cuda:0")
    P = mmf.add_noise(X, 1.0, np.inf, 0.01, 1, 5)                     # infinite OSNR: identity, powers still measured
    torch.cuda.synchronize()
    assert np.array_equal(X.cpu().numpy(), A)
    assert np.allclose(P.cpu().numpy(), (np.abs(A) ** 2).reshape(M, 2, N).sum(axis=1).mean(axis=1), rtol=1e-13)
    assert float(P[1]) == 0.0
    P1 = mmf.add_noise(X, 1.0, 10.0, 0.01, 1, 5)
    torch.cuda.synchronize()
    got = X.cpu().numpy()
    assert np.array_equal(got[2:4], A[2:4]) and not np.array_equal(got[0], A[0])
    want, _ = orc.add_noise(A, 1.0, 10.0, 0.01, 1, 5)
    assert workloads.rel_l2_per_field(got[[0, 1, 4, 5]], want[[0, 1, 4, 5]]).max() <= TOL_NOISY_FIELD
    # the same call on the same input gives the same bits (fixed summation tree, counter-based generator)
    Y = torch.from_numpy(A).to("cuda:0")
    P2 = mmf.add_noise(Y, 1.0, 10.0, 0.01, 1, 5)
    torch.cuda.synchronize()
    assert np.array_equal(Y.cpu().numpy(), got) and np.array_equal(P1.cpu().numpy(), P2.cpu().numpy())
    # argument errors
    L, vp = mmf.lib(), ctypes.c_void_p
    a, pw = vp(X.data_ptr()), vp(P.data_ptr())
    for args in ((None, M, N, 1.0, 20.0, 0.01, 1, 0, pw), (a, 0, N, 1.0, 20.0, 0.01, 1, 0, pw), (a, M, 0, 1.0, 20.0, 0.01, 1, 0, pw),
                 (a, M, N, 0.0, 20.0, 0.01, 1, 0, pw), (a, M, N, 1.0, float("nan"), 0.01, 1, 0, pw),
                 (a, M, N, 1.0, 20.0, -1.0, 1, 0, pw), (a, M, N, 1.0, 20.0, 0.01, 0, 0, pw), (a, M, N, 1.0, 20.0, 0.01, 1, 0, None)):
        assert L.mmf_add_noise(*args, None) == mmf.MMF_EINVAL, args


def test_add_noise_after_a_propagated_link(mmf, torch, orc):
    """The order of section 6: spans with the lumped amplifier, then the noise, 'before the receiver'."""
    p = workloads.problem(1, M=6, N=1 << 13, steps=4)
    A = p.field() * 8.0
    g = float(np.exp(p.alpha * p.h * 2 / 2))
    pl = mmf.Plan(p.M, p.N, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa)
    X = torch.from_numpy(A).to("cuda:0")
    pl.propagate_spans(X, 2, 2, g)
    mmf.add_noise(X, p.dt, 20.0, 0.0125, 60, 11)
    torch.cuda.synchronize()
    link = orc.rk4ip_spans(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 2, 2, g)
    want, _ = orc.add_noise(link, p.dt, 20.0, 0.0125, 60, 11)
    assert workloads.rel_l2_per_field(X.cpu().numpy(), want).max() <= 1e-10
    pl.destroy()
