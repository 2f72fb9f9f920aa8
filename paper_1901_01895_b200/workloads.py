"""Seeded synthetic workloads shaped like the paper's — shared by the oracle-side
tests and the CUDA-side tests / bench.  This module holds NONE of the method's arithmetic (no L, no N, no RK4):
only fibre-parameter draws and input waveforms.  Recipe: DESIGN.md "Input recipe".

Units everywhere: time ps, length m, power W.  So dt [ps], h [m], alpha [1/m] (linear power attenuation),
beta_n [ps^n/m], gamma [1/(W m)], |A|^2 [W].
"""
import math

import numpy as np

SEED_BASE = 190101895
LN10 = math.log(10.0)

# The five configurations of BASELINE.json (index = config id).
CONFIGS = [
    dict(name="cfg0", M=2, N=1 << 12, dt=1.0, h=100.0, steps=100, b1=5.0, b2=(-21.7, -21.7), kap=(0.1, 0.5),
         signal="qpsk_gauss", mw=1.0),
    dict(name="cfg1", M=6, N=1 << 16, dt=0.5, h=50.0, steps=1000, b1=10.0, b2=(-21.7, -21.7), kap=(0.1, 0.5),
         signal="wdm", nch=16, mw=0.5),
    dict(name="cfg2", M=36, N=1 << 18, dt=0.25, h=100.0, steps=500, b1=20.0, b2=(-23.0, -20.0), kap=(0.05, 0.6),
         signal="wdm", nch=60, mw=0.1),
    dict(name="cfg3", M=120, N=1 << 18, dt=0.25, h=250.0, steps=200, b1=50.0, b2=(-25.0, -18.0), kap=(0.01, 0.5),
         signal="wdm", nch=8, mw=0.1),
    dict(name="cfg4", M=120, N=1 << 22, dt=0.0625, h=250.0, steps=50, b1=50.0, b2=(-25.0, -18.0), kap=(0.01, 0.5),
         signal="noise", band_thz=1.5, mw=1.0),
]

ALPHA_DB_KM = 0.2       # dB/km
BETA3_PS3_KM = 0.1      # ps^3/km
GAMMA_W_KM = 1.3        # 1/(W km)
BAUD_PER_PS = 0.032     # 32 GBd
SPACING_PER_PS = 0.05   # 50 GHz
ROLLOFF = 0.1


class Problem:
    """Plain container: sizes, fibre parameters (SI-ish units above) and a row-wise input generator."""

    def __init__(self, cfg, M, N, steps):
        c = CONFIGS[cfg]
        self.cfg, self.name = cfg, c["name"]
        self.M, self.N, self.steps = int(M), int(N), int(steps)
        self.R = 2 * self.M
        self.dt, self.h = float(c["dt"]), float(c["h"])
        self.alpha = ALPHA_DB_KM * LN10 / 10.0 / 1000.0
        self.gamma = GAMMA_W_KM / 1000.0
        self.K = 4
        rng = np.random.default_rng([SEED_BASE, cfg, 0])
        b1 = rng.uniform(-c["b1"], c["b1"], size=self.M) / 1000.0
        lo, hi = c["b2"]
        b2 = (rng.uniform(lo, hi, size=self.M) if lo != hi else np.full(self.M, lo)) / 1000.0
        self.beta = np.zeros((self.M, self.K))
        self.beta[:, 1] = b1
        self.beta[:, 2] = b2
        self.beta[:, 3] = BETA3_PS3_KM / 1000.0
        klo, khi = c["kap"]
        U = rng.uniform(klo, khi, size=(self.M, self.M))
        kap = np.triu(U, 1)
        self.kappa = np.ascontiguousarray(kap + kap.T + np.eye(self.M))
        self._c = c

    def kappa_general(self, seed=0):
        """A [2M][2M] per-polarisation coupling matrix for this config: the config's mode-pair
        strengths kappa_ab, same-polarisation coupling 1 and cross-polarisation 2/3 (the ratio of a linearly
        birefringent fibre), and a seeded +-10 % spread per entry, so the matrix is NOT symmetric."""
        rng = np.random.default_rng([SEED_BASE, self.cfg, 7, int(seed)])
        pol = np.array([[1.0, 2.0 / 3.0], [2.0 / 3.0, 1.0]])
        k2 = np.kron(self.kappa, pol)
        return np.ascontiguousarray(k2 * rng.uniform(0.9, 1.1, size=k2.shape))

    def kappa_grouped(self, seed=0):
        """A mode-group kappa (Table 2: the modes form strongly coupled groups; a graded-index fibre's
        group g holds g spatial modes, 1 + 2 + ... + 15 = 120): kappa_ab = K[g(a)][g(b)] with K symmetric, unit diagonal
        and seeded off-diagonals from the config's range — every mode of a group has the same row.
        Returns (kappa [M][M], group_of [M])."""
        rng = np.random.default_rng([SEED_BASE, self.cfg, 11, int(seed)])
        group_of, g = [], 0
        while len(group_of) < self.M:
            group_of += [g] * (g + 1)
            g += 1
        group_of = np.array(group_of[:self.M])
        G = int(group_of.max()) + 1
        klo, khi = self._c["kap"]
        U = np.triu(rng.uniform(klo, khi, size=(G, G)), 1)
        K = U + U.T + np.eye(G)
        return np.ascontiguousarray(K[np.ix_(group_of, group_of)]), group_of

    # ---- input waveforms -------------------------------------------------------------------------------
    def row(self, r):
        """Input samples of field r = 2a+p (complex128, length N), seeded per row."""
        c, N = self._c, self.N
        rng = np.random.default_rng([SEED_BASE, self.cfg, 1, int(r)])
        kind = c["signal"]
        if kind == "qpsk_gauss":
            x = self._qpsk_gauss(rng)
            ptot = c["mw"] * 1e-3 / 2.0          # per polarisation: mean(P_a) = mw per mode
        elif kind == "wdm":
            x = self._wdm(rng, c["nch"])
            ptot = c["nch"] * c["mw"] * 1e-3 / 2.0   # per channel per mode = both polarisations together
        else:
            x = self._noise(rng, c["band_thz"])
            ptot = c["mw"] * 1e-3 / 2.0
        p = float(np.mean(x.real ** 2 + x.imag ** 2))
        return x * math.sqrt(ptot / p)

    def field(self):
        A = np.empty((self.R, self.N), dtype=np.complex128)
        for r in range(self.R):
            A[r] = self.row(r)
        return A

    def _qpsk(self, rng, n):
        b = rng.integers(0, 2, size=(2, n)) * 2 - 1
        return (b[0] + 1j * b[1]) / math.sqrt(2.0)

    def _qpsk_gauss(self, rng, sps=16, sigma=4.0):
        N = self.N
        nsym = max(1, N // sps)
        s = self._qpsk(rng, nsym)
        x = np.zeros(N, dtype=np.complex128)
        x[(np.arange(nsym) * sps) % N] = s
        t = np.arange(N)
        t = np.minimum(t, N - t).astype(np.float64)
        g = np.exp(-0.5 * (t / sigma) ** 2)
        return np.fft.ifft(np.fft.fft(x) * np.fft.fft(g))      # circular Gaussian pulse shaping

    def _wdm(self, rng, nch):
        N, dt = self.N, self.dt
        nsym = max(4, int(math.floor(N * dt * BAUD_PER_PS)))   # whole symbols per window -> periodic waveform
        rs = nsym / (N * dt)                                    # realised symbol rate [1/ps]
        # keep only channels whose band fits the simulated window (matters for shrunken test sizes)
        fmax = 0.5 / dt
        X = np.zeros(N, dtype=np.complex128)
        kk = np.fft.fftfreq(N, d=1.0 / N).astype(np.int64)      # signed bin index
        f = kk / (N * dt)
        for ch in range(nch):
            fc = (ch - (nch - 1) / 2.0) * SPACING_PER_PS
            if abs(fc) + 0.5 * (1 + ROLLOFF) * rs >= fmax:
                continue
            S = np.fft.fft(self._qpsk(rng, nsym))
            sh = int(round(fc * N * dt))
            fb = (kk - sh) / (N * dt)                           # baseband frequency of each bin for this channel
            a = np.abs(fb)
            H = np.where(a <= 0.5 * (1 - ROLLOFF) * rs, 1.0,
                         np.where(a <= 0.5 * (1 + ROLLOFF) * rs,
                                  0.5 * (1 + np.cos(np.pi / (ROLLOFF * rs) * (a - 0.5 * (1 - ROLLOFF) * rs))), 0.0))
            X += H * S[np.mod(kk - sh, nsym)]
        if not np.any(X):
            X[1] = 1.0
        return np.fft.ifft(X)

    def _noise(self, rng, band_thz):
        N, dt = self.N, self.dt
        nb = int(math.floor(band_thz * N * dt))                 # bins with |f| <= band (f in 1/ps = THz)
        nb = max(1, min(nb, N // 2 - 1))
        X = np.zeros(N, dtype=np.complex128)
        g = rng.standard_normal(2 * (2 * nb + 1))
        z = g[0::2] + 1j * g[1::2]
        X[: nb + 1] = z[: nb + 1]
        X[N - nb:] = z[nb + 1:]
        return np.fft.ifft(X)


def problem(cfg, M=None, N=None, steps=None):
    """Config `cfg` of BASELINE.json, optionally shrunk (same recipe, dt, h and parameter ranges)."""
    c = CONFIGS[cfg]
    return Problem(cfg, c["M"] if M is None else M, c["N"] if N is None else N,
                   c["steps"] if steps is None else steps)


def rel_l2_per_field(x, ref):
    """Per-row relative L2 error ||x_r - ref_r|| / max(||ref_r||, 1e-300).  Comparator only."""
    x = np.asarray(x)
    ref = np.asarray(ref)
    num = np.sqrt(np.sum(np.abs(x - ref) ** 2, axis=-1))
    den = np.maximum(np.sqrt(np.sum(np.abs(ref) ** 2, axis=-1)), 1e-300)
    return num / den
