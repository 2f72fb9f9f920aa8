"""Host-side checks of the C ABI (no GPU): the library loads, exports every symbol include/mmf.h declares, and the
argument validation that precedes any CUDA call returns MMF_EINVAL."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def mmf():
    from paper_1901_01895_b200 import build, binding
    build.build()
    return binding


def test_library_exports_every_declared_symbol(mmf):
    hdr = open(os.path.join(ROOT, "include", "mmf.h")).read()
    declared = set(re.findall(r"\b(mmf_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(mmf.SYMBOLS), declared ^ set(mmf.SYMBOLS)
    L = mmf.lib()
    for s in declared:
        assert hasattr(L, s), s
    ph = open(os.path.join(ROOT, "include", "mmf_probes.h")).read()
    probes = set(re.findall(r"\b(mmf_[a-z0-9_]+)\s*\(", ph))
    assert probes == set(mmf.PROBE_SYMBOLS), probes ^ set(mmf.PROBE_SYMBOLS)
    PL = mmf.probes_lib()
    for s in probes:
        assert hasattr(PL, s) and not hasattr(L, s), s       # the product library carries the product only
    assert L.mmf_version().startswith(b"mmf-b200")
    assert L.mmf_status_string(mmf.MMF_EINVAL) == b"invalid argument"


def test_create_rejects_bad_arguments_before_touching_cuda(mmf):
    ok = dict(M=2, N=4096, dt=1.0, h=100.0, alpha=0.0, beta=np.zeros((2, 4)), K=4, gamma=1e-3, kappa=np.eye(2))
    bad = [dict(N=4000), dict(N=8), dict(N=1 << 25), dict(M=0), dict(K=0), dict(K=9), dict(dt=0.0), dict(dt=-1.0),
           dict(h=float("nan")), dict(gamma=float("inf")), dict(beta=None), dict(kappa=None),
           dict(kappa=np.array([[1.0, np.nan], [0.0, 1.0]]))]
    for b in bad:
        kw = dict(ok)
        kw.update(b)
        rc, h = mmf.raw_create(kw["M"], kw["N"], kw["dt"], kw["h"], kw["alpha"], kw["beta"], kw["K"], kw["gamma"],
                               kw["kappa"])
        assert rc == mmf.MMF_EINVAL and not h.value, b
    L = mmf.lib()
    assert L.mmf_plan_workspace_bytes(None) == 0
    assert L.mmf_plan_destroy(None) == mmf.MMF_EINVAL
    assert L.mmf_propagate(None, None, 1, None) == mmf.MMF_EINVAL
    assert L.mmf_plan_launch_count(None) == 0


def test_missing_library_fails_loudly(mmf, monkeypatch):
    monkeypatch.setattr(mmf, "_lib", None)
    monkeypatch.setattr(mmf, "LIB_PATH", "/nonexistent/libmmf_b200.so")
    with pytest.raises(mmf.MmfError):
        mmf.lib()


def test_static_entry_point_validates_before_touching_cuda(mmf):
    """mmf_apply_nonlinear_static (the entry point that allocates nothing): argument and size checks come before any
    CUDA call, so they can be exercised without a GPU (the pointers are never dereferenced on these paths)."""
    import ctypes
    L = mmf.lib()
    fake = ctypes.c_void_p(4096)
    assert L.mmf_apply_nonlinear_static(129, 4096, 1.0, 1.0, fake, fake, fake, None) == mmf.MMF_ETOOBIG
    assert L.mmf_apply_nonlinear_static(1, (1 << 19) + 1, 1.0, 1.0, fake, fake, fake, None) == mmf.MMF_ETOOBIG
    assert L.mmf_apply_nonlinear_static(1 << 30, 1 << 40, 1.0, 1.0, fake, fake, fake, None) == mmf.MMF_ETOOBIG
    assert b"MMF_STATIC_SCRATCH_BYTES" in L.mmf_status_string(mmf.MMF_ETOOBIG)
    assert L.mmf_apply_nonlinear_static(0, 16, 1.0, 1.0, fake, fake, fake, None) == mmf.MMF_EINVAL
    assert L.mmf_apply_nonlinear_static(2, 16, 1.0, float("inf"), fake, fake, fake, None) == mmf.MMF_EINVAL
    assert L.mmf_apply_nonlinear_static(2, 16, 1.0, 1.0, fake, ctypes.c_void_p(4104), fake, None) == mmf.MMF_EINVAL
    assert L.mmf_apply_nonlinear_static(2, 16, 1.0, 1.0, fake, None, fake, None) == mmf.MMF_EINVAL
    hdr = open(os.path.join(ROOT, "include", "mmf.h")).read()
    assert int(re.search(r"#define MMF_STATIC_SCRATCH_BYTES \((\d+)u << (\d+)\)", hdr).group(1)) << 20 == mmf.STATIC_SCRATCH_BYTES


def test_shard_plan_that_cannot_run_its_apply_kernel_is_refused_at_creation(mmf):
    """A shard plan whose kappa rows + tiles exceed one SM's shared memory (include/mmf.h states the bound) must fail in
    mmf_plan_create_shard, not at the first mmf_shard_apply in the middle of a step."""
    import ctypes
    L = mmf.lib()
    dp = ctypes.POINTER(ctypes.c_double)
    for M_local, M_total in ((120, 240), (80, 240)):
        MP = (M_local + 3) & ~3
        assert 8 * (M_total * MP + 32 * M_total + 32 * MP) > 227 * 1024
        h = ctypes.c_void_p()
        beta = np.zeros((M_local, 1))
        kap = np.ones((M_local, M_total))
        rc = L.mmf_plan_create_shard(ctypes.byref(h), M_local, M_total, 0, 4096, 1.0, 1.0, 0.0, beta.ctypes.data_as(dp), 1,
                                     1.0, kap.ctypes.data_as(dp))
        assert rc == mmf.MMF_EINVAL and not h.value
