"""Host-side checks of the seeded synthetic workloads (no method arithmetic involved)."""
import numpy as np
import pytest

from paper_1901_01895_b200 import workloads


@pytest.mark.parametrize("cfg,N", [(0, 4096), (1, 1 << 13), (2, 1 << 14), (3, 1 << 13), (4, 1 << 14)])
def test_power_band_and_determinism(cfg, N):
    p = workloads.problem(cfg, M=min(workloads.CONFIGS[cfg]["M"], 4), N=N)
    A = p.field()
    assert A.shape == (2 * p.M, N) and A.dtype == np.complex128
    assert np.array_equal(A[1], p.row(1))                                  # seeded per row
    c = workloads.CONFIGS[cfg]
    per_mode = np.mean(np.abs(A[0::2]) ** 2 + np.abs(A[1::2]) ** 2, axis=1)
    want = c["mw"] * 1e-3 * (c.get("nch", 1))
    assert np.allclose(per_mode, want, rtol=1e-12)
    X = np.abs(np.fft.fft(A, axis=1)) ** 2
    assert X[:, N // 2].max() <= 1e-20 * X.max()                            # band-limited: nothing at Nyquist
    # parameters: kappa symmetric with unit diagonal, off-diagonal in range
    k = p.kappa
    assert np.array_equal(k, k.T) and np.all(np.diag(k) == 1.0)
    off = k[~np.eye(p.M, dtype=bool)]
    assert off.min() >= c["kap"][0] and off.max() <= c["kap"][1]
    assert np.all(np.abs(p.beta[:, 1]) <= c["b1"] / 1000.0)
    assert abs(p.alpha - 4.605170185988092e-05) < 1e-18


def test_full_size_shapes():
    for cfg, (M, N, steps) in enumerate([(2, 4096, 100), (6, 65536, 1000), (36, 1 << 18, 500), (120, 1 << 18, 200),
                                         (120, 1 << 22, 50)]):
        c = workloads.CONFIGS[cfg]
        assert (c["M"], c["N"], c["steps"]) == (M, N, steps)


def test_rel_l2_per_field():
    x = np.array([[3 + 4j, 0], [0, 0]], dtype=complex)
    r = workloads.rel_l2_per_field(x * (1 + 1e-3), x)
    assert abs(r[0] - 1e-3) < 1e-15 and r[1] == 0.0
