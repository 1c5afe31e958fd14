"""CPU-only: libargus.so builds for sm_100a, loads, and exports every symbol include/argus.h
declares (no compute calls without a GPU)."""
import ctypes
import os
import re

from paper_2606_20374_b200 import argus as A

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "argus.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(argus_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported():
    lib = A.load()
    names = _declared()
    assert "argus_ingest" in names and "argus_aggregate" in names
    assert "argus_phase_times" in names and "argus_diagnose" in names
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(A.EXPORTS) == names


def test_sizes_and_pure_host_calls():
    lib = A.load()
    cfg = A.ArgusConfig(4096, 1, 4096, 16, 0, 1, 0, 0)
    assert lib.argus_record_bytes(ctypes.byref(cfg)) == 64 + 32 * 17 + 160 * 4096 == 655968
    assert lib.argus_table_bytes(ctypes.byref(cfg)) == 655968 * 4096
    assert lib.argus_record_bytes(None) == 0
    assert lib.argus_strerror(0) == b"ok" and b"invalid" in lib.argus_strerror(-1)
    assert b"sm_100a" in lib.argus_version()
    assert ctypes.sizeof(A.ArgusConfig) == 40 and ctypes.sizeof(A.ArgusDiagOut) == 48
    for dt, n in ((A.EVENT_DTYPE, 32), (A.CELL_DTYPE, 160), (A.SPAN_DTYPE, 32), (A.STAT_DTYPE, 32),
                  (A.HEADER_DTYPE, 64)):
        assert dt.itemsize == n


def test_create_rejects_bad_config_without_touching_cuda():
    lib = A.load()
    h = ctypes.c_void_p()
    for cfg in (A.ArgusConfig(0, 1, 1, 1, 0, 0, 0, 0), A.ArgusConfig(1, 0, 1, 1, 0, 0, 0, 0),
                A.ArgusConfig(1, 1, 0, 1, 0, 0, 0, 0), A.ArgusConfig(1, 1, 1, 0, 0, 0, 0, 0),
                A.ArgusConfig(1, 1, 1, 65, 0, 0, 0, 0), A.ArgusConfig(16385, 1, 1, 1, 0, 0, 0, 0)):
        assert lib.argus_create(ctypes.byref(cfg), None, 0, ctypes.byref(h)) == A.EINVAL
        assert lib.argus_workspace_bytes(ctypes.byref(cfg)) == 0
    assert lib.argus_create(None, None, 0, ctypes.byref(h)) == A.EINVAL
    assert lib.argus_workspace_bytes(None) == 0
    for cfg in (A.ArgusConfig(16384, 1 << 20, 1, 1, 0, 0, 0, 0),        # R*T >= 2^31
                A.ArgusConfig(1, 1, 1 << 25, 1, 0, 0, 0, 0),            # record >= 4 GiB
                A.ArgusConfig(2, 4, 2, 1, 0xFFFFFFFE, 0, 0, 0),         # step_base + T wraps (R19)
                A.ArgusConfig(1, 1 << 12, 1 << 20, 1, 0, 0, 0, 0)):     # more series than one grid
        assert lib.argus_create(ctypes.byref(cfg), None, 0, ctypes.byref(h)) == A.ESIZE
    ok = A.ArgusConfig(2, 4, 2, 1, 0xFFFFFFFC, 0, 0, 0)                 # step_base + T == 2^32 is fine
    assert lib.argus_create(ctypes.byref(ok), ctypes.c_void_p(128), 1 << 30, ctypes.byref(h)) == A.EINVAL  # misaligned workspace
    assert lib.argus_destroy(None) == A.EINVAL
    assert lib.argus_aggregate(None, None, 0, None, None) == A.EINVAL


def test_no_cpu_fallback():
    """Without a CUDA device argus_create must fail loudly (never compute on the host)."""
    import torch
    if torch.cuda.is_available():
        return
    lib = A.load()
    h = ctypes.c_void_p()
    cfg = A.ArgusConfig(2, 1, 2, 1, 0, 1, 0, 0)
    assert lib.argus_create(ctypes.byref(cfg), None, 0, ctypes.byref(h)) in (A.ECUDA, A.ENOMEM)
    assert not h.value
    import pytest
    with pytest.raises(A.ArgusError):
        A.Argus(2, 1, 2, 1)
