"""Thin Python binding of the C ABI in include/mmf.h (argument marshalling only — every step of the path runs in
the CUDA kernels of libmmf_b200.so).  PyTorch is used for device buffers and streams, nothing else.

There is no CPU fallback: if the CUDA library is missing or cannot be loaded, importing a symbol from here raises.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmmf_b200.so")

MMF_OK, MMF_EINVAL, MMF_ENOMEM, MMF_ECUDA, MMF_ETOOBIG = 0, -1, -2, -3, -4
STATIC_SCRATCH_BYTES = 4 << 20   # MMF_STATIC_SCRATCH_BYTES of include/mmf.h

# every symbol include/mmf.h declares (tests check that the built library exports all of them)
SYMBOLS = ["mmf_plan_create", "mmf_plan_create_general", "mmf_plan_create_shard", "mmf_shard_begin", "mmf_shard_powers",
           "mmf_shard_apply", "mmf_shard_linear", "mmf_shard_end", "mmf_plan_workspace_bytes", "mmf_plan_set_workspace", "mmf_propagate", "mmf_propagate_ssfm",
           "mmf_propagate_ssfm_agrawal", "mmf_propagate_spans",
           "mmf_propagate_host", "mmf_propagate_host_batch", "mmf_apply_linear", "mmf_apply_nonlinear", "mmf_debug_forward",
           "mmf_debug_freq_index", "mmf_plan_launch_count", "mmf_plan_groups", "mmf_plan_set_timing", "mmf_kernel_class_count",
           "mmf_kernel_class_name", "mmf_plan_get_timing", "mmf_plan_destroy", "mmf_status_string", "mmf_version",
           "mmf_apply_nonlinear_static", "mmf_add_noise", "mmf_debug_noise_words"]

# every symbol include/mmf_probes.h declares (libmmf_probes.so: measurement probes, not part of the product library)
PROBE_SYMBOLS = ["mmf_probe_fp64", "mmf_probe_tma_copy", "mmf_probe_onchip"]
PROBES_LIB_PATH = os.path.join(_HERE, "libmmf_probes.so")

_lib = None
_probes = None


class MmfError(RuntimeError):
    pass


def lib():
    """Load libmmf_b200.so (built in-tree by paper_1901_01895_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise MmfError("CUDA library %s is missing: run `python -m paper_1901_01895_b200.build` "
                       "(there is no CPU fallback)" % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    vp, ll, i, d, sz = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    dp = ctypes.POINTER(ctypes.c_double)
    L.mmf_plan_create.argtypes = [ctypes.POINTER(vp), i, ll, d, d, d, dp, i, d, dp]
    L.mmf_plan_create.restype = i
    L.mmf_plan_create_general.argtypes = [ctypes.POINTER(vp), i, ll, d, d, d, dp, i, d, dp]
    L.mmf_plan_create_general.restype = i
    L.mmf_plan_create_shard.argtypes = [ctypes.POINTER(vp), i, i, i, ll, d, d, d, dp, i, d, dp]
    L.mmf_plan_create_shard.restype = i
    L.mmf_shard_begin.argtypes = [vp, vp, vp]
    L.mmf_shard_begin.restype = i
    L.mmf_shard_powers.argtypes = [vp, i, vp, ll, ll, vp]
    L.mmf_shard_powers.restype = i
    L.mmf_shard_apply.argtypes = [vp, i, vp, ll, ll, d, vp]
    L.mmf_shard_apply.restype = i
    L.mmf_shard_linear.argtypes = [vp, i, vp]
    L.mmf_shard_linear.restype = i
    L.mmf_shard_end.argtypes = [vp, vp]
    L.mmf_shard_end.restype = i
    L.mmf_plan_workspace_bytes.argtypes = [vp]
    L.mmf_plan_workspace_bytes.restype = sz
    L.mmf_plan_set_workspace.argtypes = [vp, vp, sz, vp]
    L.mmf_plan_set_workspace.restype = i
    L.mmf_propagate.argtypes = [vp, vp, i, vp]
    L.mmf_propagate.restype = i
    L.mmf_propagate_ssfm.argtypes = [vp, vp, i, vp]
    L.mmf_propagate_ssfm.restype = i
    L.mmf_propagate_spans.argtypes = [vp, vp, i, i, d, vp]
    L.mmf_propagate_spans.restype = i
    L.mmf_propagate_ssfm_agrawal.argtypes = [vp, vp, i, i, vp]
    L.mmf_propagate_ssfm_agrawal.restype = i
    L.mmf_propagate_host.argtypes = [vp, vp, vp, i, vp]
    L.mmf_propagate_host.restype = i
    L.mmf_propagate_host_batch.argtypes = [vp, ctypes.POINTER(vp), i, vp, vp, i, vp]
    L.mmf_propagate_host_batch.restype = i
    L.mmf_apply_linear.argtypes = [vp, vp, vp]
    L.mmf_apply_linear.restype = i
    L.mmf_apply_nonlinear.argtypes = [vp, vp, vp, vp]
    L.mmf_apply_nonlinear.restype = i
    L.mmf_debug_forward.argtypes = [vp, vp, vp, vp]
    L.mmf_debug_forward.restype = i
    L.mmf_debug_freq_index.argtypes = [vp, ctypes.POINTER(ll)]
    L.mmf_debug_freq_index.restype = i
    L.mmf_plan_groups.argtypes = [vp]
    L.mmf_plan_groups.restype = i
    L.mmf_plan_launch_count.argtypes = [vp]
    L.mmf_plan_launch_count.restype = ll
    L.mmf_plan_set_timing.argtypes = [vp, i]
    L.mmf_plan_set_timing.restype = i
    L.mmf_kernel_class_count.argtypes = []
    L.mmf_kernel_class_count.restype = i
    L.mmf_kernel_class_name.argtypes = [i]
    L.mmf_kernel_class_name.restype = ctypes.c_char_p
    L.mmf_plan_get_timing.argtypes = [vp, i, dp, ctypes.POINTER(ll), dp]
    L.mmf_plan_get_timing.restype = i
    L.mmf_plan_destroy.argtypes = [vp]
    L.mmf_plan_destroy.restype = i
    L.mmf_status_string.argtypes = [i]
    L.mmf_status_string.restype = ctypes.c_char_p
    L.mmf_apply_nonlinear_static.argtypes = [i, ll, d, d, vp, vp, vp, vp]
    L.mmf_apply_nonlinear_static.restype = i
    L.mmf_add_noise.argtypes = [vp, i, ll, d, d, d, i, ctypes.c_ulonglong, vp, vp]
    L.mmf_add_noise.restype = i
    L.mmf_debug_noise_words.argtypes = [ctypes.c_ulonglong, ctypes.c_uint, ctypes.c_ulonglong, ll, vp, vp]
    L.mmf_debug_noise_words.restype = i
    L.mmf_version.argtypes = []
    L.mmf_version.restype = ctypes.c_char_p
    _lib = L
    return L


def probes_lib():
    """Load libmmf_probes.so (bench.py --probes).  Fails loudly if absent."""
    global _probes
    if _probes is not None:
        return _probes
    if not os.path.exists(PROBES_LIB_PATH):
        raise MmfError("probe library %s is missing: run `python -m paper_1901_01895_b200.build`" % PROBES_LIB_PATH)
    L = ctypes.CDLL(PROBES_LIB_PATH)
    i, d, sz, vp, ll = ctypes.c_int, ctypes.c_double, ctypes.c_size_t, ctypes.c_void_p, ctypes.c_longlong
    dp = ctypes.POINTER(ctypes.c_double)
    ull, u = ctypes.c_ulonglong, ctypes.c_uint
    L.mmf_probe_fp64.argtypes = [i, i, i, dp, dp]
    L.mmf_probe_fp64.restype = i
    L.mmf_probe_onchip.argtypes = [i, i, i, dp, dp]
    L.mmf_probe_onchip.restype = i
    L.mmf_probe_tma_copy.argtypes = [vp, sz, ull, ull, ull, u, u, i, i, i, i, ll, i, i, i, dp, dp]
    L.mmf_probe_tma_copy.restype = i
    _probes = L
    return L


def _check(rc, what):
    if rc != MMF_OK:
        raise MmfError("%s failed: %s (%d)" % (what, lib().mmf_status_string(rc).decode(), rc))


def _stream_ptr(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


class Plan:
    """mmf_plan_create / mmf_plan_set_workspace / mmf_propagate / mmf_plan_destroy with torch-owned buffers."""

    def __init__(self, M, N, dt, h, alpha, beta, gamma, kappa, device="cuda:0", general=False, shard=None):
        """general=True: kappa is the [2M][2M] per-polarisation matrix (mmf_plan_create_general).
        shard=(M_total, mode0): a row-shard plan (mmf_plan_create_shard): M own modes, kappa = their [M][M_total] rows."""
        import torch
        L = lib()
        self.M, self.N = int(M), int(N)
        beta = np.ascontiguousarray(beta, dtype=np.float64).reshape(self.M, -1)
        kd = 2 * self.M if general else self.M
        kc = int(shard[0]) if shard is not None else kd
        kappa = np.ascontiguousarray(kappa, dtype=np.float64).reshape(kd, kc)
        self._h = ctypes.c_void_p()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        dp = ctypes.POINTER(ctypes.c_double)
        if shard is not None:
            self.M_total, self.mode0 = int(shard[0]), int(shard[1])
            rc = L.mmf_plan_create_shard(ctypes.byref(self._h), self.M, self.M_total, self.mode0, self.N, float(dt), float(h),
                                         float(alpha), beta.ctypes.data_as(dp), beta.shape[1], float(gamma),
                                         kappa.ctypes.data_as(dp))
        else:
            create = L.mmf_plan_create_general if general else L.mmf_plan_create
            rc = create(ctypes.byref(self._h), self.M, self.N, float(dt), float(h), float(alpha),
                        beta.ctypes.data_as(dp), beta.shape[1], float(gamma), kappa.ctypes.data_as(dp))
        _check(rc, "mmf_plan_create")
        nbytes = L.mmf_plan_workspace_bytes(self._h)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-self.workspace.data_ptr()) % 256
        self._ws_ptr = self.workspace.data_ptr() + off
        _check(L.mmf_plan_set_workspace(self._h, ctypes.c_void_p(self._ws_ptr), nbytes, _stream_ptr()),
               "mmf_plan_set_workspace")

    # -- helpers -------------------------------------------------------------------------------------------
    def _field_ptr(self, A):
        import torch
        assert A.is_cuda and A.dtype == torch.complex128 and A.is_contiguous()
        assert tuple(A.shape) == (2 * self.M, self.N), (A.shape, self.M, self.N)
        return ctypes.c_void_p(A.data_ptr())

    # -- the C ABI -------------------------------------------------------------------------------------------
    def propagate(self, A, nsteps, stream=None):
        """A: torch complex128 CUDA tensor (2M, N), advanced in place by nsteps RK4IP steps."""
        _check(lib().mmf_propagate(self._h, self._field_ptr(A), int(nsteps), _stream_ptr(stream)), "mmf_propagate")
        return A

    def propagate_spans(self, A, nspans, steps_per_span, gain, stream=None):
        """nspans spans of steps_per_span RK4IP steps, the lumped amplifier A <- gain * A after each span."""
        _check(lib().mmf_propagate_spans(self._h, self._field_ptr(A), int(nspans), int(steps_per_span), float(gain),
                                         _stream_ptr(stream)), "mmf_propagate_spans")
        return A

    def propagate_ssfm(self, A, nsteps, stream=None):
        """In-place SSFM-RK4 propagation (symmetric split step, Eq. 4) of a CUDA complex128 tensor [2M, N]."""
        _check(lib().mmf_propagate_ssfm(self._h, self._field_ptr(A), int(nsteps), _stream_ptr(stream)),
               "mmf_propagate_ssfm")

    def propagate_ssfm_agrawal(self, A, nsteps, niter=2, stream=None):
        """In-place SSFM-Agrawal propagation (symmetric split step, iterative trapezoidal nonlinear part)."""
        _check(lib().mmf_propagate_ssfm_agrawal(self._h, self._field_ptr(A), int(nsteps), int(niter),
                                                _stream_ptr(stream)), "mmf_propagate_ssfm_agrawal")

    # -- row-sharded propagation: the stage calls paper_1901_01895_b200/sharded.py sequences around its all-gather
    def shard_begin(self, A, stream=None):
        _check(lib().mmf_shard_begin(self._h, self._field_ptr(A), _stream_ptr(stream)), "mmf_shard_begin")

    def _chunk_ptr(self, P, t_count):
        import torch
        assert P.is_cuda and P.dtype == torch.float64 and P.is_contiguous()
        assert tuple(P.shape) == (self.M_total, t_count), (tuple(P.shape), self.M_total, t_count)
        return ctypes.c_void_p(P.data_ptr())

    def shard_powers(self, stage, P, t_first=0, t_count=None, stream=None):
        """P: CUDA float64 [M_total][t_count], the power block of samples t_first .. t_first + t_count - 1."""
        t_count = self.N if t_count is None else int(t_count)
        _check(lib().mmf_shard_powers(self._h, int(stage), self._chunk_ptr(P, t_count), int(t_first), t_count,
                                      _stream_ptr(stream)), "mmf_shard_powers")

    def shard_apply(self, stage, P, t_first=0, t_count=None, gain=1.0, stream=None):
        t_count = self.N if t_count is None else int(t_count)
        _check(lib().mmf_shard_apply(self._h, int(stage), self._chunk_ptr(P, t_count), int(t_first), t_count, float(gain),
                                     _stream_ptr(stream)), "mmf_shard_apply")

    def shard_linear(self, which, stream=None):
        _check(lib().mmf_shard_linear(self._h, int(which), _stream_ptr(stream)), "mmf_shard_linear")

    def shard_end(self, stream=None):
        _check(lib().mmf_shard_end(self._h, _stream_ptr(stream)), "mmf_shard_end")

    def propagate_host(self, A_host, A_scratch, nsteps, stream=None):
        """A_host: pinned torch complex128 CPU tensor (2M, N); A_scratch: CUDA tensor of the same shape."""
        import torch
        assert (not A_host.is_cuda) and A_host.dtype == torch.complex128 and A_host.is_contiguous()
        assert tuple(A_host.shape) == (2 * self.M, self.N)
        _check(lib().mmf_propagate_host(self._h, ctypes.c_void_p(A_host.data_ptr()), self._field_ptr(A_scratch),
                                        int(nsteps), _stream_ptr(stream)), "mmf_propagate_host")
        return A_host

    def propagate_host_batch(self, hosts, scratch0, scratch1, nsteps, stream=None):
        """hosts: list of pinned torch complex128 CPU tensors (2M, N); scratch0 / scratch1: CUDA tensors of that shape."""
        import torch
        for H in hosts:
            assert (not H.is_cuda) and H.dtype == torch.complex128 and H.is_contiguous()
            assert tuple(H.shape) == (2 * self.M, self.N)
        arr = (ctypes.c_void_p * len(hosts))(*[H.data_ptr() for H in hosts])
        _check(lib().mmf_propagate_host_batch(self._h, arr, len(hosts), self._field_ptr(scratch0),
                                              self._field_ptr(scratch1) if scratch1 is not None else None, int(nsteps),
                                              _stream_ptr(stream)), "mmf_propagate_host_batch")
        return hosts

    def apply_linear(self, X, stream=None):
        _check(lib().mmf_apply_linear(self._h, self._field_ptr(X), _stream_ptr(stream)), "mmf_apply_linear")
        return X

    def apply_nonlinear(self, U, OUT, stream=None):
        _check(lib().mmf_apply_nonlinear(self._h, self._field_ptr(U), self._field_ptr(OUT), _stream_ptr(stream)),
               "mmf_apply_nonlinear")
        return OUT

    def debug_forward(self, X, SPEC, stream=None):
        _check(lib().mmf_debug_forward(self._h, self._field_ptr(X), self._field_ptr(SPEC), _stream_ptr(stream)),
               "mmf_debug_forward")
        return SPEC

    def debug_freq_index(self):
        idx = np.empty(self.N, dtype=np.int64)
        _check(lib().mmf_debug_freq_index(self._h, idx.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong))),
               "mmf_debug_freq_index")
        return idx

    def groups(self):
        """Number of distinct kappa rows the grouped contraction runs on (0: dense)."""
        return int(lib().mmf_plan_groups(self._h))

    def launch_count(self):
        return int(lib().mmf_plan_launch_count(self._h))

    def set_timing(self, enable):
        _check(lib().mmf_plan_set_timing(self._h, 1 if enable else 0), "mmf_plan_set_timing")

    def get_timing(self):
        """[{name, total_ms, launches, alg_bytes_per_launch}] for every kernel class with at least one launch."""
        L = lib()
        out = []
        for k in range(L.mmf_kernel_class_count()):
            ms, n, by = ctypes.c_double(), ctypes.c_longlong(), ctypes.c_double()
            _check(L.mmf_plan_get_timing(self._h, k, ctypes.byref(ms), ctypes.byref(n), ctypes.byref(by)),
                   "mmf_plan_get_timing")
            if n.value:
                out.append(dict(name=L.mmf_kernel_class_name(k).decode(), total_ms=ms.value, launches=n.value,
                                alg_bytes_per_launch=by.value))
        return out

    def destroy(self):
        if self._h:
            lib().mmf_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def apply_nonlinear_static(kappa, U, OUT, h, gamma, stream=None):
    """mmf_apply_nonlinear_static: OUT <- h N(U) U for callers that may not allocate device memory (no plan, no
    workspace; the mode powers go through the library's fixed 4 MiB static device array, so M * N <= 524288).
    kappa: CUDA float64 tensor [M][M]; U, OUT: CUDA complex128 tensors [2M][N] (OUT may be U).  All three are the
    caller's; this wrapper only passes their addresses and raises MmfError on a non-zero status (MMF_ETOOBIG when the
    problem exceeds the static array).  The first call on a device does the one-time set-up: see include/mmf.h."""
    import torch
    assert kappa.is_cuda and kappa.dtype == torch.float64 and kappa.is_contiguous() and kappa.dim() == 2
    M = kappa.shape[0]
    assert kappa.shape[1] == M
    for T in (U, OUT):
        assert T.is_cuda and T.dtype == torch.complex128 and T.is_contiguous() and T.shape[0] == 2 * M
    assert U.shape == OUT.shape
    _check(lib().mmf_apply_nonlinear_static(int(M), int(U.shape[1]), float(h), float(gamma),
                                            ctypes.c_void_p(kappa.data_ptr()), ctypes.c_void_p(U.data_ptr()),
                                            ctypes.c_void_p(OUT.data_ptr()), _stream_ptr(stream)),
           "mmf_apply_nonlinear_static")
    return OUT


def add_noise(A, dt, osnr_db, ref_bw, nch, seed, mode_power=None, stream=None):
    """mmf_add_noise: noise loading in place on the CUDA complex128 tensor A [2M][N].  Returns the CUDA
    float64 tensor [M] of the mode powers measured before the noise (allocated here with torch unless passed in)."""
    import torch
    assert A.is_cuda and A.dtype == torch.complex128 and A.is_contiguous() and A.dim() == 2 and A.shape[0] % 2 == 0
    M = A.shape[0] // 2
    if mode_power is None:
        mode_power = torch.empty(M, dtype=torch.float64, device=A.device)
    assert mode_power.is_cuda and mode_power.dtype == torch.float64 and mode_power.numel() == M
    _check(lib().mmf_add_noise(ctypes.c_void_p(A.data_ptr()), int(M), int(A.shape[1]), float(dt), float(osnr_db),
                               float(ref_bw), int(nch), int(seed), ctypes.c_void_p(mode_power.data_ptr()),
                               _stream_ptr(stream)), "mmf_add_noise")
    return mode_power


def noise_words(seed, row, t0, count, device="cuda:0", stream=None):
    """mmf_debug_noise_words: CUDA int32 tensor [count][4] holding the Philox output words (as uint32 bit patterns)."""
    import torch
    out = torch.empty((int(count), 4), dtype=torch.int32, device=device)
    _check(lib().mmf_debug_noise_words(int(seed), int(row), int(t0), int(count), ctypes.c_void_p(out.data_ptr()),
                                       _stream_ptr(stream)), "mmf_debug_noise_words")
    return out


def raw_create(M, N, dt, h, alpha, beta, K, gamma, kappa, general=False):
    """mmf_plan_create(_general) with raw arguments (for error-path tests).  Returns (status, handle)."""
    h_ = ctypes.c_void_p()
    dp = ctypes.POINTER(ctypes.c_double)
    b = None if beta is None else np.ascontiguousarray(beta, dtype=np.float64).ctypes.data_as(dp)
    k = None if kappa is None else np.ascontiguousarray(kappa, dtype=np.float64).ctypes.data_as(dp)
    create = lib().mmf_plan_create_general if general else lib().mmf_plan_create
    rc = create(ctypes.byref(h_), int(M), int(N), float(dt), float(h), float(alpha), b, int(K), float(gamma), k)
    return rc, h_


def probe_fp64(kind, threads=512, iters=4000):
    """mmf_probe_fp64: (ms per launch, thread-level (kind 5: warp-level) instructions per launch)."""
    ms, n = ctypes.c_double(), ctypes.c_double()
    _check(probes_lib().mmf_probe_fp64(int(kind), int(threads), int(iters), ctypes.byref(ms), ctypes.byref(n)), "mmf_probe_fp64")
    return ms.value, n.value


def probe_onchip(kind, threads=512, iters=2000):
    """mmf_probe_onchip: (ms per launch, clock64 ticks per operation with every warp of the CTA running the loop)."""
    ms, clk = ctypes.c_double(), ctypes.c_double()
    _check(probes_lib().mmf_probe_onchip(int(kind), int(threads), int(iters), ctypes.byref(ms), ctypes.byref(clk)),
           "mmf_probe_onchip")
    return ms.value, clk.value


def probe_tma_copy(buf, dim0, dim1, stride_bytes, box0, box1, nbox, nct_log, c0_mul, c1_mul, ntiles, slots=3, bulk=0,
                   reps=3):
    """mmf_probe_tma_copy over the torch uint8 CUDA tensor `buf`: (ms per launch, bytes moved read + write)."""
    ms, by = ctypes.c_double(), ctypes.c_double()
    _check(probes_lib().mmf_probe_tma_copy(ctypes.c_void_p(buf.data_ptr()), buf.numel(), int(dim0), int(dim1), int(stride_bytes),
                                    int(box0), int(box1), int(nbox), int(nct_log), int(c0_mul), int(c1_mul), int(ntiles),
                                    int(slots), int(bulk), int(reps), ctypes.byref(ms), ctypes.byref(by)),
           "mmf_probe_tma_copy")
    return ms.value, by.value
