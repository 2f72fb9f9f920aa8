"""Pins of the oracle's general per-polarisation coupling (Fig. 2: "Storing all
kappa values requires a matrix of 2M x 2M elements"): out_r = i h gamma (sum_s kappa2[r][s] |u_s|^2) u_r.
  * exact integer arithmetic (numpy int64, written separately) with a random NON-symmetric integer 2M x 2M matrix;
  * the Manakov special case kappa2[2a+p][2b+q] = kappa_ab must reproduce the M x M routine bit for bit on integers;
  * alpha = beta = 0: every |A_r|^2 is conserved and the exact flow is A_r exp(i gamma sum_s kappa2[r][s] |A_s|^2 z):
    the RK4IP step converges to it with order 4 (x16 per halving);
  * the whole of Eq. (1) with this N against an independent adaptive integration (scipy DOP853), order 4;
  * the packed size the paper prints: (2M 2M)/2 + M = 28 920 entries at M = 120 (tests/golden/paper_sizes.txt).
"""
import math

import numpy as np


def rel(x, ref):
    return float(np.linalg.norm(np.ravel(x - ref)) / max(np.linalg.norm(np.ravel(ref)), 1e-300))


def rand_c(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def test_general_nonlinear_integer_exact(orc):
    for M, N in ((1, 4), (3, 16), (4, 8), (37, 8)):
        rng = np.random.default_rng(M * 100 + N)
        R = 2 * M
        ur = rng.integers(-30, 31, size=(R, N))
        ui = rng.integers(-30, 31, size=(R, N))
        k2 = rng.integers(-9, 10, size=(R, R))
        P = ur * ur + ui * ui                      # int64
        S = k2 @ P                                 # int64, exact
        want = (-S * ui) + 1j * (S * ur)           # (i S) (ur + i ui)
        got = orc.nonlinear_general((ur + 1j * ui).astype(complex), 1.0, k2.astype(float))
        assert np.array_equal(got, want.astype(complex))


def test_manakov_is_the_special_case(orc):
    M, N = 5, 16
    rng = np.random.default_rng(9)
    u = (rng.integers(-20, 21, size=(2 * M, N)) + 1j * rng.integers(-20, 21, size=(2 * M, N))).astype(complex)
    kap = rng.integers(-7, 8, size=(M, M)).astype(float)
    k2 = np.kron(kap, np.ones((2, 2)))             # kappa2[2a+p][2b+q] = kappa_ab
    assert np.array_equal(orc.nonlinear_general(u, 1.0, k2), orc.nonlinear(u, 1.0, kap))


def test_general_phase_rotation_fourth_order(orc):
    M, N = 2, 16
    rng = np.random.default_rng(12)
    A = rand_c(rng, 2 * M, N) * np.array([1.0, 0.4, 0.8, 1.3])[:, None]
    k2 = rng.uniform(0.1, 1.0, size=(2 * M, 2 * M))          # non-symmetric, polarisations unequal
    gamma, z = 0.8, 0.2
    want = A * np.exp(1j * gamma * (k2 @ np.abs(A) ** 2) * z)
    errs = [rel(orc.rk4ip_general(A, 1.0, z / n, 0.0, np.zeros((M, 1)), gamma, k2, n, nthreads=1), want)
            for n in (2, 4, 8, 16)]
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert errs[-1] < 1e-5
    assert all(12.0 < r < 20.0 for r in ratios[1:]), (errs, ratios)


def test_general_fourth_order_against_independent_solution_of_eq1(orc):
    from scipy.integrate import solve_ivp
    M, N, dt, z = 2, 64, 1.0, 60.0
    rng = np.random.default_rng(81)
    X = np.zeros((2 * M, N), dtype=complex)
    X[:, :4] = rand_c(rng, 2 * M, 4)
    X[:, -3:] = rand_c(rng, 2 * M, 3)
    A0 = np.fft.ifft(X, axis=1) * (N / 16) * np.array([6.0, 2.5, 4.4, 7.0])[:, None]
    alpha, gamma = 2e-3, 1.7e-3
    beta = np.array([[4e-3, 9e-3, -25e-3, 3e-3], [-6e-3, -7e-3, -18e-3, -2e-3]])
    k2 = rng.uniform(0.2, 1.0, size=(2 * M, 2 * M))
    w = 2 * np.pi * np.fft.fftfreq(N, d=dt)
    Lsym = np.empty((2 * M, N), dtype=complex)
    for r in range(2 * M):
        L = np.full(N, -alpha / 2.0, dtype=complex)
        for n, b in enumerate(beta[r // 2]):
            L = L + 1j * (1j ** n) / math.factorial(n) * b * (1j * w) ** n     # Eq. (1) as printed, d/dt -> i w
        Lsym[r] = L

    def rhs(_z, y):
        A = (y[: y.size // 2] + 1j * y[y.size // 2:]).reshape(2 * M, N)
        d = (np.fft.ifft(Lsym * np.fft.fft(A, axis=1), axis=1) + 1j * gamma * (k2 @ np.abs(A) ** 2) * A).ravel()
        return np.concatenate([d.real, d.imag])

    y0 = np.concatenate([A0.ravel().real, A0.ravel().imag])
    sol = solve_ivp(rhs, (0.0, z), y0, method="DOP853", rtol=1e-12, atol=1e-14)
    assert sol.success
    ref = (sol.y[: y0.size // 2, -1] + 1j * sol.y[y0.size // 2:, -1]).reshape(2 * M, N)
    errs = [rel(orc.rk4ip_general(A0, dt, z / n, alpha, beta, gamma, k2, n, nthreads=1), ref) for n in (8, 16, 32)]
    assert errs[-1] < 1e-6, errs
    assert 11.0 < errs[0] / errs[1] < 21.0 and 11.0 < errs[1] / errs[2] < 21.0, errs
    # and it differs from the Manakov reduction of the same matrix (the polarisation structure matters)
    kap = k2[0::2, 0::2]
    assert rel(orc.rk4ip(A0, dt, z / 32, alpha, beta, gamma, kap, 32, nthreads=1), ref) > 1e-3


def test_packed_size_the_paper_prints():
    M = 120
    assert (2 * M * 2 * M) // 2 + M == 28920                  # PAPER.md:176 "(2M 2M)/2 + M", :182 "28920"


# ------------------------------------------------------------------------------- spans with lumped amplifiers
def test_spans_gamma_zero_loss_is_compensated_exactly(orc):
    """gamma = 0, gain = exp(alpha L_span / 2): after every span the spectrum has its input magnitude back and the
    field is the lossless linear solution over the whole link (closed form written with numpy)."""
    M, N, dt, h, k, nsp = 2, 64, 0.7, 3.0, 4, 3
    rng = np.random.default_rng(14)
    X = rand_c(rng, 2 * M, N)
    X[:, N // 2] = 0
    A = np.fft.ifft(X, axis=1)
    alpha = 0.05
    beta = np.array([[0.01, 0.03, -0.05, 0.004], [-0.02, -0.01, -0.03, 0.002]])
    w = 2 * np.pi * np.fft.fftfreq(N, d=dt)
    want = np.empty_like(A)
    for r in range(2 * M):
        L = np.zeros(N, dtype=complex)
        for n, b in enumerate(beta[r // 2]):
            L = L + 1j * (1j ** n) / math.factorial(n) * b * (1j * w) ** n
        want[r] = np.fft.ifft(np.exp(L * h * k * nsp) * np.fft.fft(A[r]))        # alpha = 0 over the whole link
    got = orc.rk4ip_spans(A, dt, h, alpha, beta, 0.0, np.eye(M), nsp, k, math.exp(alpha * h * k / 2), nthreads=1)
    assert rel(got, want) <= 1e-13
    assert abs(np.sum(np.abs(got) ** 2) / np.sum(np.abs(A) ** 2) - 1.0) <= 1e-13


def test_spans_amplifier_acts_between_spans_not_inside(orc):
    """with nonlinearity the place of the gain matters: gain after each span differs from one gain at the end (same
    total gain) and from no gain — and equals propagating span by span with the amplitude scaled in between."""
    M, N, dt, h, k = 2, 32, 1.0, 2.0, 3
    rng = np.random.default_rng(15)
    A = rand_c(rng, 2 * M, N) * 0.6
    beta = np.array([[0.0, 0.01, -0.02, 0.001], [0.0, -0.01, -0.03, 0.001]])
    kappa = np.array([[1.0, 0.4], [0.7, 1.0]])
    alpha, gamma, g = 0.05, 0.05, 1.3
    got = orc.rk4ip_spans(A, dt, h, alpha, beta, gamma, kappa, 2, k, g, nthreads=1)
    by_hand = orc.rk4ip(orc.rk4ip(A, dt, h, alpha, beta, gamma, kappa, k, nthreads=1) * g, dt, h, alpha, beta, gamma,
                        kappa, k, nthreads=1) * g
    assert np.array_equal(got, by_hand)
    end_only = orc.rk4ip(A, dt, h, alpha, beta, gamma, kappa, 2 * k, nthreads=1) * g * g
    assert rel(got, end_only) > 1e-3
    assert np.array_equal(orc.rk4ip_spans(A, dt, h, alpha, beta, gamma, kappa, 0, k, g), A)
