"""Pins for the CPU oracle (oracle/rk4ip_oracle.cpp) against what the paper and the mathematics fix.

None of these tests re-type the oracle's own formulae and compare them with themselves: each expected value
comes from (i) the definition of the DFT / an independent library FFT, (ii) a closed-form solution of Eq. (1)
 in a special case, (iii) an invariant of Eq. (1), (iv) an independent adaptive integrator
(scipy DOP853) applied to Eq. (1) *as printed in the time domain* with spectral differentiation, (v) exact
integer arithmetic, or (vi) numbers the paper prints (tests/golden/paper_sizes.txt).
"""
import math
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def rel(x, ref):
    return float(np.linalg.norm(np.ravel(x - ref)) / max(np.linalg.norm(np.ravel(ref)), 1e-300))


def rand_c(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


# ------------------------------------------------------------------------------------------------- P1: transforms
@pytest.mark.parametrize("N", [2, 4, 8, 16, 32, 64])
@pytest.mark.parametrize("sign", [1, -1])
def test_fft_equals_direct_dft(orc, N, sign):
    """radix-2 FFT == the plain O(N^2) Fourier sum (definition of the DFT)."""
    x = rand_c(np.random.default_rng(N + sign), N)
    assert rel(orc.fft(x, sign), orc.dft(x, sign)) <= 1e-14


def test_direct_dft_matches_written_out_sum(orc):
    """The O(N^2) routine itself against the sum written with numpy's exp (N = 5 and 12: also non powers of 2)."""
    for N in (5, 12):
        x = rand_c(np.random.default_rng(N), N)
        k = np.arange(N)[:, None]
        n = np.arange(N)[None, :]
        for sign in (1, -1):
            want = (np.exp(sign * 2j * np.pi * k * n / N) * x[None, :]).sum(axis=1)
            assert rel(orc.dft(x, sign), want) <= 1e-14


@pytest.mark.parametrize("N", [8, 256, 4096, 1 << 15])
def test_fft_equals_library_fft(orc, N):
    """Against numpy's pocketfft (an independent library): sign -1 is numpy's forward, sign +1 is N * ifft."""
    x = rand_c(np.random.default_rng(7 * N), N)
    assert rel(orc.fft(x, -1), np.fft.fft(x)) <= 5e-15
    assert rel(orc.fft(x, +1), N * np.fft.ifft(x)) <= 5e-15
    assert rel(orc.fft(orc.fft(x, +1), -1) / N, x) <= 5e-15          # round trip


def test_fft_sign_and_exactness_on_deltas(orc):
    """sign=+1 of a delta at n=1 is exp(+2 pi i k/N): for N=4 exactly (1, i, -1, -i) — bit-exact (Gaussian ints)."""
    out = orc.fft(np.array([0, 1, 0, 0], dtype=complex), +1)
    assert np.array_equal(out, np.array([1, 1j, -1, -1j]))
    out = orc.fft(np.array([0, 1, 0, 0], dtype=complex), -1)
    assert np.array_equal(out, np.array([1, -1j, -1, 1j]))
    x = np.array([3 + 2j, -1 + 5j, 4 - 7j, -6 - 1j])
    F = np.array([[1, 1, 1, 1], [1, 1j, -1, -1j], [1, -1, 1, -1], [1, -1j, -1, 1j]])
    assert np.array_equal(orc.fft(x, +1), F @ x)


def test_omega_grid(orc):
    """w_k = 2 pi k'/(N dt), negative for k >= N/2 (reading R7) — numpy's fftfreq uses the same fold."""
    N, dt = 16, 0.25
    w = orc.omega(N, dt)
    assert np.allclose(w, 2 * np.pi * np.fft.fftfreq(N, d=dt), rtol=1e-15, atol=0)
    assert w[N // 2] < 0


# ------------------------------------------------------------------------- P2-P4, P6b: the linear operator of Eq. 1
def eq1_linear_symbol(w_np, alpha, beta_a):
    """L of Eq. (1) AS PRINTED (time domain): -alpha/2 + i sum_n (i^n/n!) beta_n d^n/dt^n, acting on exp(+i w t),
    i.e. d/dt -> (i w).  w_np are numpy-convention bin frequencies (x(t) = sum X_k exp(+i w_k t))."""
    L = np.full(w_np.shape, -alpha / 2.0, dtype=complex)
    for n, b in enumerate(beta_a):
        L = L + 1j * (1j ** n) / math.factorial(n) * b * (1j * w_np) ** n
    return L


def test_tone_eigenvalue(orc):
    """A(t) = exp(-i W t) is an eigenfunction of Eq. (1)'s L with eigenvalue -alpha/2 + i sum beta_n W^n/n!
    (apply d/dt -> -iW by hand: i^n (-iW)^n = W^n).  gamma = 0, so RK4IP must give exp(h L) exactly.  All of
    beta_0..beta_3 non-zero pins every sign and the 1/n!."""
    M, N, dt, h = 1, 64, 0.5, 37.0
    alpha = 3e-3
    beta = np.array([[0.011, -0.023, 0.017, -0.0041]])
    t = np.arange(N) * dt
    for j in (0, 1, 5, -3, -31, N // 2):
        W = 2 * np.pi * (j if j != N // 2 else -N // 2) / (N * dt)
        A = np.vstack([np.exp(-1j * W * t), 0.5j * np.exp(-1j * W * t)])
        lam = -alpha / 2 + 1j * sum(beta[0, n] * W ** n / math.factorial(n) for n in range(4))
        out = orc.rk4ip(A, dt, h, alpha, beta, 0.0, np.ones((1, 1)), 3, nthreads=1)
        assert rel(out, np.exp(3 * h * lam) * A) <= 1e-13


def test_beta1_delays(orc):
    """Only beta_1 != 0 with beta_1 h = m dt: Eq. (1) is dA/dz = -beta_1 dA/dt, so A(z,t) = A(0, t - beta_1 z):
    the samples move to LATER times (np.roll by +m); the advanced copy must fail."""
    M, N, dt, h, m = 2, 128, 0.5, 10.0, 3
    rng = np.random.default_rng(4)
    A = rand_c(rng, 2 * M, N)
    beta = np.zeros((M, 2))
    beta[:, 1] = m * dt / h
    out = orc.rk4ip(A, dt, h, 0.0, beta, 0.0, np.eye(M), 1, nthreads=1)
    assert rel(out, np.roll(A, m, axis=1)) <= 1e-13
    assert rel(out, np.roll(A, -m, axis=1)) > 0.5


def test_linear_propagation_matches_spectral_solution_of_eq1(orc):
    """gamma = 0: every k_i vanishes and Eq. (6) reduces to exp(hL).  Expected value: Eq. (1) as
    printed, solved with numpy's FFT and spectral differentiation (independent sign convention and library)."""
    M, N, dt, h, steps = 3, 256, 0.25, 55.0, 7
    rng = np.random.default_rng(11)
    X = rand_c(rng, 2 * M, N)
    X[:, N // 2] = 0            # the Nyquist bin's frequency sign is a convention (reading R7; pinned by the tone test)
    A = np.fft.ifft(X, axis=1)
    alpha = 4.6e-5
    beta = rng.uniform(-1, 1, size=(M, 4)) * np.array([0.01, 0.02, 0.02, 0.002])
    out = orc.rk4ip(A, dt, h, alpha, beta, 0.0, np.eye(M), steps, nthreads=2)
    w = 2 * np.pi * np.fft.fftfreq(N, d=dt)
    want = np.empty_like(A)
    for r in range(2 * M):
        want[r] = np.fft.ifft(np.fft.fft(A[r]) * np.exp(steps * h * eq1_linear_symbol(w, alpha, beta[r // 2])))
    assert rel(out, want) <= 1e-13


def test_energy_decays_as_exp_minus_alpha_z(orc):
    """gamma = 0, alpha > 0: sum |A|^2 = exp(-alpha z) E0 exactly (the dispersive part is unitary)."""
    M, N, dt, h, steps = 2, 128, 1.0, 100.0, 5
    rng = np.random.default_rng(5)
    A = rand_c(rng, 2 * M, N)
    alpha = 0.2 * math.log(10) / 10 / 1000
    beta = np.array([[0, 1e-3, -21.7e-3, 1e-4]] * M)
    out = orc.rk4ip(A, dt, h, alpha, beta, 0.0, np.eye(M), steps, nthreads=1)
    e0, e1 = np.sum(np.abs(A) ** 2), np.sum(np.abs(out) ** 2)
    assert abs(e1 / e0 - math.exp(-alpha * h * steps)) <= 1e-13


# ------------------------------------------------------------------------------------ P5: the nonlinear operator
def test_nonlinear_phase_rotation_exact_solution(orc):
    """alpha = beta = 0: every time sample obeys dA_a/dz = i gamma (sum_b kappa_ab P_b) A_a with P conserved, so
    A_a(z) = A_a(0) exp(i gamma S_a z).  kappa NON-symmetric (catches a transposed kappa), polarisations with
    different powers (catches mis-pairing).  RK4IP is then plain RK4: error falls x16 per halving."""
    M, N, dt = 3, 32, 1.0
    rng = np.random.default_rng(9)
    A = rand_c(rng, 2 * M, N) * np.array([1.0, 0.3, 0.7, 1.4, 0.2, 0.9])[:, None]
    kappa = rng.uniform(0.1, 1.0, size=(M, M))
    gamma, z = 0.9, 0.15
    P = (np.abs(A[0::2]) ** 2 + np.abs(A[1::2]) ** 2)
    S = kappa @ P
    want = A * np.exp(1j * gamma * np.repeat(S, 2, axis=0) * z)
    beta = np.zeros((M, 1))
    errs = []
    for n in (4, 8, 16, 32):
        out = orc.rk4ip(A, dt, z / n, 0.0, beta, gamma, kappa, n, nthreads=1)
        errs.append(rel(out, want))
        Pout = np.abs(out[0::2]) ** 2 + np.abs(out[1::2]) ** 2
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert errs[-1] < 1e-5
    assert all(12.0 < r < 20.0 for r in ratios[1:]), ratios
    assert rel(Pout, P) < 1e-6                      # power per mode conserved to the method's order


def test_nonlinear_operator_integer_exact(orc):
    """Gaussian-integer u, integer non-symmetric kappa, h*gamma = 1: every product and sum is exact in fp64, so the
    oracle must equal int64 arithmetic BIT FOR BIT:  out = i * (sum_b kappa_ab (|u_bx|^2+|u_by|^2)) * u."""
    M, N = 5, 17
    rng = np.random.default_rng(3)
    ur = rng.integers(-30, 31, size=(2 * M, N))
    ui = rng.integers(-30, 31, size=(2 * M, N))
    kap = rng.integers(-9, 10, size=(M, M))
    P = ur[0::2] ** 2 + ui[0::2] ** 2 + ur[1::2] ** 2 + ui[1::2] ** 2
    S = np.repeat(kap @ P, 2, axis=0)
    want = (-S * ui) + 1j * (S * ur)
    got = orc.nonlinear(ur + 1j * ui, 1.0, kap.astype(float))
    assert np.array_equal(got, want.astype(complex))


# --------------------------------------------------------------------------------- P6a: energy with alpha = 0
def test_energy_conservation_drift_is_fourth_order(orc):
    """alpha = 0: Eq. (1) conserves sum_r sum_t |A|^2 (L is skew, N is a phase).  RK4IP conserves it only to
    the method's order: the drift must shrink ~x16 (global 4th order) per halving."""
    M, N, dt, z = 2, 64, 1.0, 300.0
    rng = np.random.default_rng(21)
    X = np.zeros((2 * M, N), dtype=complex)
    X[:, :6] = rand_c(rng, 2 * M, 6)
    X[:, -5:] = rand_c(rng, 2 * M, 5)
    A = np.fft.ifft(X, axis=1) * 40
    beta = np.array([[0, 2e-3, -21.7e-3, 1e-4], [0, -2e-3, -20e-3, 1e-4]])
    kappa = np.array([[1.0, 0.4], [0.4, 1.0]])
    e0 = np.sum(np.abs(A) ** 2)
    drift = []
    for n in (16, 32, 64):
        out = orc.rk4ip(A, dt, z / n, 0.0, beta, 2e-4, kappa, n, nthreads=1)
        drift.append(abs(np.sum(np.abs(out) ** 2) / e0 - 1))
    assert drift[-1] < 1e-6
    assert 10 < drift[0] / drift[1] < 40 and 10 < drift[1] / drift[2] < 40, drift


# ------------------------------------------------------------------------------------------------- P7: soliton
def test_fundamental_soliton_keeps_shape(orc):
    """Single mode, y = 0, beta_2 < 0, A = sqrt(P0) sech(t/T0) with gamma P0 T0^2/|beta_2| = 1 (textbook, ref [6]
    of the paper): A(z) = A(0) exp(i gamma P0 z / 2).  Error x16 per halving; y stays exactly 0."""
    N, dt, T0 = 1024, 0.5, 10.0
    b2, gamma = -21.7e-3, 1.3e-3
    P0 = abs(b2) / (gamma * T0 ** 2)
    z = T0 ** 2 / abs(b2)                      # one dispersion length: phase 0.5 rad
    t = (np.arange(N) - N // 2) * dt
    A = np.vstack([math.sqrt(P0) / np.cosh(t / T0), np.zeros(N)]).astype(complex)
    want = A * np.exp(0.5j * gamma * P0 * z)
    beta = np.array([[0.0, 0.0, b2]])
    errs = []
    for n in (4, 8, 16, 32):
        out = orc.rk4ip(A, dt, z / n, 0.0, beta, gamma, np.ones((1, 1)), n, nthreads=1)
        errs.append(rel(out[0], want[0]))
        assert np.all(out[1] == 0)
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert errs[-1] < 2e-7, errs
    assert all(13.0 < r < 18.0 for r in ratios[1:]), ratios


# ------------------------------------------------- P8: the whole of Eq. (1) against an independent integrator
def test_converges_at_fourth_order_to_independent_solution_of_eq1(orc):
    """Eq. (1) as printed (time-domain operators, spectral differentiation with numpy's FFT), integrated by scipy's
    adaptive DOP853 at rtol 1e-12.  RK4IP must approach it with err(h)/err(h/2) -> 16 ("globally fourth-order
    accurate").  Non-symmetric kappa, all of alpha, beta_0..beta_3, gamma non-zero, per-mode betas,
    unequal polarisation powers: a dropped term, wrong sign, transposed kappa or mis-paired polarisation fails."""
    from scipy.integrate import solve_ivp
    M, N, dt, z = 2, 128, 1.0, 120.0
    rng = np.random.default_rng(77)
    X = np.zeros((2 * M, N), dtype=complex)
    X[:, :4] = rand_c(rng, 2 * M, 4)           # narrow band: four-wave mixing must not reach the Nyquist bin, whose
    X[:, -3:] = rand_c(rng, 2 * M, 3)          # frequency sign is a convention (reading R7)
    A0 = np.fft.ifft(X, axis=1) * (N / 32) * np.array([9.0, 3.6, 6.6, 10.5])[:, None]
    alpha, gamma = 2e-3, 1.7e-3
    beta = np.array([[4e-3, 9e-3, -25e-3, 3e-3], [-6e-3, -7e-3, -18e-3, -2e-3]])
    kappa = np.array([[1.0, 0.35], [0.8, 0.6]])
    w = 2 * np.pi * np.fft.fftfreq(N, d=dt)
    Lsym = np.vstack([eq1_linear_symbol(w, alpha, beta[r // 2]) for r in range(2 * M)])

    def rhs(_z, y):
        A = (y[: y.size // 2] + 1j * y[y.size // 2:]).reshape(2 * M, N)
        lin = np.fft.ifft(Lsym * np.fft.fft(A, axis=1), axis=1)
        P = np.abs(A[0::2]) ** 2 + np.abs(A[1::2]) ** 2
        d = lin + 1j * gamma * np.repeat(kappa @ P, 2, axis=0) * A
        d = d.ravel()
        return np.concatenate([d.real, d.imag])

    y0 = np.concatenate([A0.ravel().real, A0.ravel().imag])
    sol = solve_ivp(rhs, (0.0, z), y0, method="DOP853", rtol=1e-12, atol=1e-14)
    assert sol.success
    ref = (sol.y[: y0.size // 2, -1] + 1j * sol.y[y0.size // 2:, -1]).reshape(2 * M, N)
    assert rel(ref, A0) > 0.3                                   # the problem is not trivial
    errs = []
    for n in (16, 32, 64, 128):
        out = orc.rk4ip(A0, dt, z / n, alpha, beta, gamma, kappa, n, nthreads=1)
        errs.append(rel(out, ref))
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert errs[-1] < 1e-9, errs
    assert all(12.0 < r < 20.0 for r in ratios), (errs, ratios)


# ------------------------------------------------------------------------------------------- P9: composition
def test_composition_is_bit_identical(orc):
    from paper_1901_01895_b200 import workloads
    p = workloads.problem(0, N=512, steps=5)
    A = p.field()
    a = orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 5, nthreads=2)
    b = orc.rk4ip(orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 2, nthreads=1),
                  p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 3, nthreads=3)
    assert np.array_equal(a, b)
    assert np.array_equal(orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 0), A)


def test_zero_field_stays_zero(orc):
    """A field that is exactly zero stays exactly zero through D and N."""
    from paper_1901_01895_b200 import workloads
    p = workloads.problem(0, N=256, steps=2)
    A = p.field()
    A[1] = 0
    out = orc.rk4ip(A, p.dt, p.h, p.alpha, p.beta, p.gamma, p.kappa, 2)
    assert np.all(out[1] == 0) and np.any(out[0] != 0)


# ------------------------------------------------------------------------------------ P11: the paper's sizes
def test_paper_printed_sizes():
    """Layout arithmetic: rows x N x bytes reproduce the MiB figures the paper prints (golden file, cited)."""
    n = 0
    for line in open(os.path.join(HERE, "golden", "paper_sizes.txt")):
        line = line.split("#")[0].split()
        if not line:
            continue
        name, rows, N, b, want = line[0], int(line[1]), int(line[2]), int(line[3]), int(line[4])
        if name.startswith("kappa_triangular"):
            assert rows * rows // 2 + rows // 2 == want
        else:
            assert rows * N * b == want * (1 << 20)
        n += 1
    assert n == 6


# ------------------------------------------------------- pins at the sizes / phases the oracle is the authority for
def test_fft_equals_library_fft_at_full_length(orc):
    """The oracle's radix-2 FFT is the authority at N = 2^22 (config 4): one row against numpy's pocketfft there."""
    N = 1 << 22
    x = rand_c(np.random.default_rng(22), N)
    assert rel(orc.fft(x, -1), np.fft.fft(x)) <= 5e-15
    assert rel(orc.fft(x, +1), N * np.fft.ifft(x)) <= 5e-15


def test_tone_eigenvalue_at_large_phase_against_mpmath(orc):
    """Config 4's dispersion phase (h/2) sum_n beta_n w^n / n! reaches ~4e3 rad at the band edge (hard
    part 1).  A tone exp(-i W t) at such bins, gamma = 0: the output must be exp(h L(W)) times the input with the
    eigenvalue computed by mpmath at 50 digits from Eq. (1)'s symbol — an fp64 evaluation of the phase would be off by
    ~1e-12 here, a sign or 1/n! slip by O(1)."""
    import mpmath as mp
    mp.mp.dps = 50
    N, dt, h, alpha = 1 << 14, 0.0625, 250.0, 4.6e-5
    beta = np.array([[1.7e-4, 4.9e-2, -2.5e-2, 1.0e-4]])
    worst_phase = 0.0
    for j in (8190, -8191, 5000, -N // 2):
        W = 2 * mp.pi * mp.mpf(j) / (mp.mpf(N) * mp.mpf(dt))
        sym = sum(mp.mpf(float(b)) * W ** n / mp.factorial(n) for n, b in enumerate(beta[0]))
        worst_phase = max(worst_phase, abs(float(sym * h / 2)))
        lam = mp.exp((-mp.mpf(alpha) / 2 + 1j * sym) * mp.mpf(h))            # one step = two exp(h/2 L)
        t = np.arange(N)
        A = np.zeros((2, N), dtype=complex)
        A[0] = np.exp(-2j * np.pi * ((j * t) % N) / N)                        # exp(-i W t), exact index reduction
        A[1] = 0.5j * A[0]
        out = orc.rk4ip(A, dt, h, alpha, beta, 0.0, np.eye(1), 1)
        want = complex(lam) * A
        assert rel(out, want) <= 2e-13, (j, rel(out, want))
    assert worst_phase > 3e3                                                   # the regime the pin is for
