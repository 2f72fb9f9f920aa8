"""ctypes loader for the CPU oracle (oracle/rk4ip_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It builds liboracle.so with g++ on first use (no CUDA, no torch) and marshals numpy arrays; there is no
arithmetic of the method in this file.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rk4ip_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force=False):
    """Compile oracle/rk4ip_oracle.cpp -> oracle/liboracle.so (plain g++, no fast-math).
    MMF_ORACLE_LIB in the environment names a library built otherwise from the same source (tests/test_oracle_sanitized.py
    runs the pins on an -fsanitize=address,undefined build); it is then loaded as it is."""
    if os.environ.get("MMF_ORACLE_LIB"):
        return os.environ["MMF_ORACLE_LIB"]
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-o", tmp, _SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ll, i, d = ctypes.c_longlong, ctypes.c_int, ctypes.c_double
        L.orc_dft.argtypes = [dp, dp, ll, i]
        L.orc_fft.argtypes = [dp, ll, i]
        L.orc_omega.argtypes = [dp, ll, d]
        L.orc_linear_table.argtypes = [dp, i, ll, d, d, d, dp, i, i]
        L.orc_apply_D.argtypes = [dp, i, ll, dp, i]
        L.orc_nonlinear.argtypes = [dp, dp, i, ll, d, dp, i]
        L.orc_rk4ip.argtypes = [dp, i, ll, d, d, d, dp, i, d, dp, i, i]
        L.orc_ssfm_rk4.argtypes = [dp, i, ll, d, d, d, dp, i, d, dp, i, i]
        L.orc_nonlinear_general.argtypes = [dp, dp, i, ll, d, dp, i]
        L.orc_rk4ip_general.argtypes = [dp, i, ll, d, d, d, dp, i, d, dp, i, i]
        L.orc_rk4ip_spans.argtypes = [dp, i, ll, d, d, d, dp, i, d, dp, i, i, i, d, i]
        L.orc_ssfm_agrawal.argtypes = [dp, i, ll, d, d, d, dp, i, d, dp, i, i, i]
        u32p = ctypes.POINTER(ctypes.c_uint32)
        L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.orc_noise_unit.argtypes = [dp, ctypes.c_ulonglong, ctypes.c_uint, ctypes.c_ulonglong, ll]
        L.orc_add_noise.argtypes = [dp, i, ll, d, d, d, i, ctypes.c_ulonglong, dp]
        L.orc_philox4x32_10.restype = L.orc_noise_unit.restype = L.orc_add_noise.restype = i
        for f in (L.orc_dft, L.orc_fft, L.orc_omega, L.orc_linear_table, L.orc_apply_D, L.orc_nonlinear,
                  L.orc_rk4ip, L.orc_ssfm_rk4, L.orc_ssfm_agrawal, L.orc_nonlinear_general, L.orc_rk4ip_general, L.orc_rk4ip_spans):
            f.restype = i
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def default_threads():
    return max(1, len(os.sched_getaffinity(0)))


def dft(x, sign):
    x = _c128(x)
    out = np.empty_like(x)
    assert lib().orc_dft(_p(x), _p(out), x.size, sign) == 0
    return out


def fft(x, sign):
    x = _c128(x).copy()
    assert lib().orc_fft(_p(x), x.size, sign) == 0
    return x


def omega(N, dt):
    w = np.empty(N, dtype=np.float64)
    assert lib().orc_omega(_p(w), N, dt) == 0
    return w


def linear_table(M, N, dt, hh, alpha, beta, nthreads=1):
    beta = _f64(beta).reshape(M, -1)
    E = np.empty((M, N), dtype=np.complex128)
    assert lib().orc_linear_table(_p(E), M, N, dt, hh, alpha, _p(beta), beta.shape[1], nthreads) == 0
    return E


def apply_D(x, E, nthreads=1):
    x = _c128(x).copy()
    E = _c128(E)
    M, N = E.shape
    assert x.shape == (2 * M, N)
    assert lib().orc_apply_D(_p(x), M, N, _p(E), nthreads) == 0
    return x


def nonlinear(u, hgamma, kappa, nthreads=1):
    u = _c128(u)
    R, N = u.shape
    M = R // 2
    kappa = _f64(kappa).reshape(M, M)
    out = np.empty_like(u)
    assert lib().orc_nonlinear(_p(u), _p(out), M, N, hgamma, _p(kappa), nthreads) == 0
    return out


def rk4ip(A, dt, h, alpha, beta, gamma, kappa, nsteps, nthreads=None, inplace=False):
    """Return A advanced nsteps RK4IP steps.  A: (2M, N) complex128; beta: (M, K); kappa: (M, M).
    inplace=True advances the caller's (contiguous complex128) array itself: one 15 GiB copy less at config 4."""
    if inplace:
        assert A.dtype == np.complex128 and A.flags.c_contiguous
    else:
        A = _c128(A).copy()
    R, N = A.shape
    M = R // 2
    assert R == 2 * M
    beta = _f64(beta).reshape(M, -1)
    kappa = _f64(kappa).reshape(M, M)
    if nthreads is None:
        nthreads = default_threads()
    rc = lib().orc_rk4ip(_p(A), M, N, dt, h, alpha, _p(beta), beta.shape[1], gamma, _p(kappa), nsteps, nthreads)
    assert rc == 0, "orc_rk4ip rejected its arguments"
    return A


def ssfm_rk4(A, dt, h, alpha, beta, gamma, kappa, nsteps, nthreads=None):
    """Return A advanced nsteps SSFM-RK4 steps (symmetric split step, Eq. 4).  Same arguments as rk4ip."""
    A = _c128(A).copy()
    R, N = A.shape
    M = R // 2
    assert R == 2 * M
    beta = _f64(beta).reshape(M, -1)
    kappa = _f64(kappa).reshape(M, M)
    if nthreads is None:
        nthreads = default_threads()
    rc = lib().orc_ssfm_rk4(_p(A), M, N, dt, h, alpha, _p(beta), beta.shape[1], gamma, _p(kappa), nsteps, nthreads)
    assert rc == 0, "orc_ssfm_rk4 rejected its arguments"
    return A


def ssfm_agrawal(A, dt, h, alpha, beta, gamma, kappa, nsteps, niter=2, nthreads=None):
    """Return A advanced nsteps SSFM-Agrawal steps (symmetric split step, iterative trapezoidal nonlinear part with
    niter iterations per step; Eq. 4, reading R14).  Same arguments as rk4ip."""
    A = _c128(A).copy()
    R, N = A.shape
    M = R // 2
    assert R == 2 * M
    beta = _f64(beta).reshape(M, -1)
    kappa = _f64(kappa).reshape(M, M)
    if nthreads is None:
        nthreads = default_threads()
    rc = lib().orc_ssfm_agrawal(_p(A), M, N, dt, h, alpha, _p(beta), beta.shape[1], gamma, _p(kappa), nsteps, niter,
                                nthreads)
    assert rc == 0, "orc_ssfm_agrawal rejected its arguments"
    return A


def nonlinear_general(u, hgamma, kappa2, nthreads=1):
    """(i hgamma sum_s kappa2[r][s] |u_s|^2) u_r with the general per-polarisation [2M][2M] coupling matrix."""
    u = _c128(u)
    R, N = u.shape
    kappa2 = _f64(kappa2).reshape(R, R)
    out = np.empty_like(u)
    assert lib().orc_nonlinear_general(_p(u), _p(out), R // 2, N, hgamma, _p(kappa2), nthreads) == 0
    return out


def rk4ip_general(A, dt, h, alpha, beta, gamma, kappa2, nsteps, nthreads=None):
    """rk4ip with kappa2: (2M, 2M), one coefficient per pair of polarisation modes."""
    A = _c128(A).copy()
    R, N = A.shape
    M = R // 2
    assert R == 2 * M
    beta = _f64(beta).reshape(M, -1)
    kappa2 = _f64(kappa2).reshape(R, R)
    if nthreads is None:
        nthreads = default_threads()
    rc = lib().orc_rk4ip_general(_p(A), M, N, dt, h, alpha, _p(beta), beta.shape[1], gamma, _p(kappa2), nsteps, nthreads)
    assert rc == 0, "orc_rk4ip_general rejected its arguments"
    return A


def rk4ip_spans(A, dt, h, alpha, beta, gamma, kappa, nspans, steps_per_span, gain, general=False, nthreads=None):
    """nspans spans of steps_per_span RK4IP steps, each followed by the lumped amplifier A <- gain * A."""
    A = _c128(A).copy()
    R, N = A.shape
    M = R // 2
    beta = _f64(beta).reshape(M, -1)
    kd = R if general else M
    kappa = _f64(kappa).reshape(kd, kd)
    if nthreads is None:
        nthreads = default_threads()
    rc = lib().orc_rk4ip_spans(_p(A), M, N, dt, h, alpha, _p(beta), beta.shape[1], gamma, _p(kappa), int(general),
                               nspans, steps_per_span, gain, nthreads)
    assert rc == 0, "orc_rk4ip_spans rejected its arguments"
    return A


def philox4x32_10(ctr, key):
    """The Philox-4x32-10 block function: 4 counter words, 2 key words -> 4 output words (uint32 arrays)."""
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    u32p = ctypes.POINTER(ctypes.c_uint32)
    assert c.size == 4 and k.size == 2
    assert lib().orc_philox4x32_10(c.ctypes.data_as(u32p), k.ctypes.data_as(u32p), out.ctypes.data_as(u32p)) == 0
    return out


def noise_unit(seed, row, t0, count):
    """The unit complex normal samples z(row, t0 .. t0 + count - 1) of the noise stream `seed` (E|z|^2 = 1)."""
    z = np.empty(count, dtype=np.complex128)
    assert lib().orc_noise_unit(_p(z), int(seed), int(row), int(t0), int(count)) == 0
    return z


def add_noise(A, dt, osnr_db, ref_bw, nch, seed):
    """Noise loading (reading R18): returns (A + noise, mean power per spatial mode before the noise)."""
    A = _c128(A).copy()
    R, N = A.shape
    M = R // 2
    P = np.empty(M, dtype=np.float64)
    rc = lib().orc_add_noise(_p(A), M, N, float(dt), float(osnr_db), float(ref_bw), int(nch), int(seed), _p(P))
    assert rc == 0, "orc_add_noise rejected its arguments"
    return A, P
