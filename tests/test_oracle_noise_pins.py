"""Pins of the oracle's noise loading ("White noise is added to the signals before the receiver, setting
the optical signal-to-noise ratio (OSNR) to 20 dB"; reading R18 in DESIGN.md) against things other than itself:
the generator's published known-answer vectors, the statistics a white circular Gaussian field must have, the
definition of the OSNR measured on the output, and exact scaling laws.  All seeds are fixed: the tests are
deterministic; the bounds are 5 standard errors of the respective estimator unless stated."""
import os

import numpy as np
import pytest
from scipy import stats

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answer_vectors_bit_exact(orc):
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        w = [int(x, 16) for x in r]
        assert list(orc.philox4x32_10(w[0:4], w[4:6])) == w[6:10]


def test_philox_is_a_bijection_of_the_counter_and_sensitive_to_every_word(orc):
    base = orc.philox4x32_10([1, 2, 3, 4], [5, 6])
    seen = {tuple(base)}
    for i in range(4):
        c = [1, 2, 3, 4]
        c[i] ^= 1
        seen.add(tuple(orc.philox4x32_10(c, [5, 6])))
    for k in ([4, 6], [5, 7]):
        seen.add(tuple(orc.philox4x32_10([1, 2, 3, 4], k)))
    assert len(seen) == 7
    # avalanche: one flipped counter bit changes about half of the 128 output bits
    flipped = orc.philox4x32_10([1, 2, 3, 5], [5, 6])
    nbits = sum(bin(int(a) ^ int(b)).count("1") for a, b in zip(base, flipped))
    assert 40 <= nbits <= 88


def test_unit_samples_are_standard_circular_gaussian_and_white(orc):
    n = 1 << 18
    z = orc.noise_unit(seed=2024, row=3, t0=0, count=n)
    se = 1.0 / np.sqrt(n)
    assert abs(z.mean()) < 5 * se                                     # zero mean (std of the mean of z = 1/sqrt(n))
    assert abs((np.abs(z) ** 2).mean() - 1.0) < 5 * se                 # E|z|^2 = 1; var(|z|^2) = 1
    assert abs(z.real.var() - 0.5) < 5 * 0.5 * np.sqrt(2.0 / n)         # each part N(0, 1/2)
    assert abs(z.imag.var() - 0.5) < 5 * 0.5 * np.sqrt(2.0 / n)
    assert abs((z * z).mean()) < 5 * se                               # circular: E z^2 = 0 (parts uncorrelated, equal variance)
    for part in (z.real, z.imag):                                      # normality: Kolmogorov-Smirnov against N(0, 1/2)
        assert stats.kstest(part / np.sqrt(0.5), "norm").pvalue > 1e-3
    assert stats.kstest(np.abs(z) ** 2, "expon").pvalue > 1e-3          # |z|^2 ~ Exp(1)
    assert stats.kstest((np.angle(z) + np.pi) / (2 * np.pi), "uniform").pvalue > 1e-3
    for lag in (1, 2, 3, 7, 64, 4097):                                  # white: no correlation between samples
        assert abs((z[lag:] * np.conj(z[:-lag])).mean()) < 5 / np.sqrt(n - lag)
    # flat spectrum: the power in each of 16 equal bands of the periodogram is 1/16 of the total
    S = np.abs(np.fft.fft(z)) ** 2
    bands = S.reshape(16, -1).sum(axis=1) / S.sum()
    assert np.abs(bands - 1 / 16).max() < 5 * (1 / 16) / np.sqrt(n / 16)
    assert np.abs(z).max() < 6.5                                       # the 52-bit uniform bounds |z| by sqrt(53 ln 2) = 6.06


def test_streams_of_different_rows_seeds_and_offsets(orc):
    n = 1 << 16
    a = orc.noise_unit(7, 0, 0, n)
    for other in (orc.noise_unit(7, 1, 0, n), orc.noise_unit(8, 0, 0, n), orc.noise_unit(7 + (1 << 32), 0, 0, n)):
        assert abs((a * np.conj(other)).mean()) < 5 / np.sqrt(n)        # uncorrelated streams
        assert not np.array_equal(a, other)
    # the sample depends on (seed, row, t) only: a window of the stream equals the stream taken at that offset,
    # also across the 32-bit boundary of the sample counter
    assert np.array_equal(orc.noise_unit(7, 0, 1000, 50), a[1000:1050])
    big = (1 << 32) - 10
    w = orc.noise_unit(7, 0, big, 20)
    assert np.array_equal(w[10:], orc.noise_unit(7, 0, 1 << 32, 10)) and not np.array_equal(w[:10], w[10:])


def test_realised_osnr_of_a_known_power_field(orc):
    """Constant-power rows with a different power per mode: measure the noise actually added and form the OSNR from
    its definition — signal power per channel over the noise power of BOTH polarisations inside the reference
    bandwidth — and compare with the request."""
    M, N, dt, ref_bw, nch, osnr_db = 3, 1 << 16, 0.0625e-12, 12.5e9, 60, 20.0
    t = np.arange(N)
    powers = np.array([1.0, 0.25, 4.0]) * 1e-3 * nch                    # W per spatial mode (both polarisations)
    A = np.empty((2 * M, N), complex)
    for a in range(M):
        A[2 * a] = np.sqrt(0.7 * powers[a]) * np.exp(2j * np.pi * 5 * t / N)
        A[2 * a + 1] = np.sqrt(0.3 * powers[a]) * np.exp(-2j * np.pi * 11 * t / N)
    out, P = orc.add_noise(A, dt, osnr_db, ref_bw, nch, seed=99)
    assert np.allclose(P, powers, rtol=1e-13)
    noise = out - A
    for a in range(M):
        var_x, var_y = (np.abs(noise[2 * a]) ** 2).mean(), (np.abs(noise[2 * a + 1]) ** 2).mean()
        assert abs(var_x / var_y - 1.0) < 5 * np.sqrt(2.0 / N)           # the same noise power in both polarisations
        psd = 0.5 * (var_x + var_y) * dt                                # W/Hz per polarisation: white over 1/dt
        osnr = (powers[a] / nch) / (2.0 * psd * ref_bw)
        assert abs(osnr / 10 ** (osnr_db / 10) - 1.0) < 5 / np.sqrt(2 * N)
        # and in the band itself: noise power inside a ref_bw-wide window of the spectrum, both polarisations
        S = (np.abs(np.fft.fft(noise[2 * a])) ** 2 + np.abs(np.fft.fft(noise[2 * a + 1])) ** 2) / N ** 2
        f = np.fft.fftfreq(N, dt)
        nb = int((np.abs(f) < 40 * ref_bw / 2).sum())                   # 40 reference bandwidths for a usable estimate
        inband = S[np.abs(f) < 40 * ref_bw / 2].sum() / 40
        assert abs((powers[a] / nch) / inband / 100.0 - 1.0) < 5 / np.sqrt(nb)


def test_noise_scaling_laws_are_exact_and_infinite_osnr_adds_nothing(orc):
    M, N, dt, ref_bw = 2, 4096, 0.5, 0.01
    rng = np.random.default_rng(5)
    A = rng.standard_normal((2 * M, N)) + 1j * rng.standard_normal((2 * M, N))
    out_inf, P = orc.add_noise(A, dt, np.inf, ref_bw, 1, seed=1)
    assert np.array_equal(out_inf, A)
    assert np.allclose(P, (np.abs(A) ** 2).reshape(M, 2, N).sum(axis=1).mean(axis=1), rtol=1e-13)
    n0 = orc.add_noise(A, dt, 10.0, ref_bw, 1, seed=1)[0] - A
    n20 = orc.add_noise(A, dt, 30.0, ref_bw, 1, seed=1)[0] - A           # 20 dB more OSNR: amplitude / 10, same stream
    assert np.allclose(n20 * 10.0, n0, rtol=1e-12, atol=1e-14)
    n4 = orc.add_noise(A, dt, 10.0, ref_bw, 4, seed=1)[0] - A            # 4 channels share the power: amplitude / 2
    assert np.allclose(n4 * 2.0, n0, rtol=1e-12, atol=1e-14)
    nb = orc.add_noise(A, dt, 10.0, 4 * ref_bw, 1, seed=1)[0] - A        # 4 x the reference bandwidth: amplitude / 2
    assert np.allclose(nb * 2.0, n0, rtol=1e-12, atol=1e-14)
    nd = orc.add_noise(A, 4 * dt, 10.0, ref_bw, 1, seed=1)[0] - A        # 4 x coarser sampling: 1/4 the band, amplitude / 2
    assert np.allclose(nd * 2.0, n0, rtol=1e-12, atol=1e-14)
    # a mode with no signal gets no noise; the others are untouched by its presence
    B = A.copy()
    B[2:4] = 0.0
    out_b = orc.add_noise(B, dt, 10.0, ref_bw, 1, seed=1)[0]
    assert np.array_equal(out_b[2:4], B[2:4]) and np.array_equal(out_b[:2] - B[:2], n0[:2])


def test_noise_of_a_row_does_not_depend_on_the_matrix_size(orc):
    """z(row, t) is a function of (seed, row, t): a larger matrix repeats the smaller one's noise on the shared part,
    and the added field is sigma_a z with sigma_a from the formula of R18."""
    dt, ref_bw, nch, osnr_db, seed = 2.0, 0.05, 3, 13.0, 77
    small = np.full((4, 64), 2.0 + 0j)
    large = np.full((10, 256), 2.0 + 0j)
    ns = orc.add_noise(small, dt, osnr_db, ref_bw, nch, seed)[0] - small
    nl = orc.add_noise(large, dt, osnr_db, ref_bw, nch, seed)[0] - large
    assert np.allclose(ns, nl[:4, :64], rtol=0, atol=1e-15)
    sigma = np.sqrt((8.0 / nch) / (2 * ref_bw * 10 ** (osnr_db / 10)) / dt)        # P_a = |2|^2 + |2|^2 = 8
    for r in range(4):
        assert np.allclose(ns[r], sigma * orc.noise_unit(seed, r, 0, 64), rtol=1e-13, atol=1e-15)
