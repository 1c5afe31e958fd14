"""ctypes wrapper of argus_oracle.c (plain single-threaded C).  TEST INFRASTRUCTURE, NOT PRODUCT."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "argus_oracle.c")
_SO = os.path.join(_HERE, "liboracle.so")

CELL_DTYPE = np.dtype([("count", "<u8"), ("sum", "<u8"), ("min", "<u8"), ("max", "<u8"),
                       ("hist", "<u4", (32,))])
SPAN_DTYPE = np.dtype([("min_start", "<i8"), ("max_end", "<i8"), ("span", "<u8"), ("n", "<u8")])
STAT_DTYPE = np.dtype([("median", "<u8"), ("mad", "<u8"), ("n_high", "<u4"), ("n_low", "<u4"),
                       ("reserved", "<u8")])
HEADER_DTYPE = np.dtype([("magic", "<u4"), ("version", "<u2"), ("n_phases", "<u2"),
                         ("n_sigs", "<u4"), ("rank", "<u4"), ("step", "<u4"), ("reserved0", "<u4"),
                         ("n_events", "<u8"), ("min_start", "<i8"), ("max_end", "<i8"),
                         ("iter_ns", "<u8"), ("reserved1", "<u8")])
assert CELL_DTYPE.itemsize == 160 and SPAN_DTYPE.itemsize == 32
assert STAT_DTYPE.itemsize == 32 and HEADER_DTYPE.itemsize == 64

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no vectoriser flags beyond the default)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.run(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-o", _SO, _SRC], check=True)
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, u32, u64 = ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64
        lib.oracle_create.restype = vp
        lib.oracle_create.argtypes = [u32, u32, u32, u32, u32]
        lib.oracle_destroy.argtypes = [vp]
        lib.oracle_aggregate.argtypes = [vp, vp, u64]
        lib.oracle_phase_times.argtypes = [vp]
        lib.oracle_record_bytes.restype = u64
        lib.oracle_record_bytes.argtypes = [vp]
        lib.oracle_encode_records.argtypes = [vp, vp]
        lib.oracle_cells.restype = vp
        lib.oracle_cells.argtypes = [vp]
        lib.oracle_spans.restype = vp
        lib.oracle_spans.argtypes = [vp]
        lib.oracle_n_valid.restype = u64
        lib.oracle_n_valid.argtypes = [vp]
        lib.oracle_n_invalid.restype = u64
        lib.oracle_n_invalid.argtypes = [vp]
        lib.oracle_bucket.restype = u32
        lib.oracle_bucket.argtypes = [u64]
        lib.oracle_series.argtypes = [vp, u32, vp, vp]
        lib.oracle_diagnose.argtypes = [vp] * 7
        _lib = lib
    return _lib


def bucket(d: int) -> int:
    return int(_load().oracle_bucket(d))


def series(x):
    """One series of u64 values -> (median, mad, n_high, n_low, flags[R])."""
    x = np.ascontiguousarray(x, dtype=np.uint64)
    stat = np.zeros(1, dtype=STAT_DTYPE)
    flags = np.zeros(x.size, dtype=np.uint8)
    _load().oracle_series(x.ctypes.data, x.size, stat.ctypes.data, flags.ctypes.data)
    s = stat[0]
    return int(s["median"]), int(s["mad"]), int(s["n_high"]), int(s["n_low"]), flags


class Oracle:
    """State of one accumulation: cells [R][T][S], spans [R][T][P+1]."""

    def __init__(self, n_ranks, n_steps, n_sigs, n_phases, step_base=0):
        self.R, self.T, self.S, self.P = n_ranks, n_steps, n_sigs, n_phases
        self.step_base = step_base
        self._lib = _load()
        self._st = self._lib.oracle_create(n_ranks, n_steps, n_sigs, n_phases, step_base)
        if not self._st:
            raise MemoryError("oracle_create")

    def __del__(self):
        if getattr(self, "_st", None):
            self._lib.oracle_destroy(self._st)
            self._st = None

    def aggregate(self, events: np.ndarray) -> None:
        """events: any array whose bytes are 32-byte records (structured or uint8)."""
        ev = np.ascontiguousarray(events)
        assert ev.nbytes % 32 == 0
        self._lib.oracle_aggregate(self._st, ev.ctypes.data, ev.nbytes // 32)

    def phase_times(self) -> None:
        self._lib.oracle_phase_times(self._st)

    @property
    def n_valid(self) -> int:
        return int(self._lib.oracle_n_valid(self._st))

    @property
    def n_invalid(self) -> int:
        return int(self._lib.oracle_n_invalid(self._st))

    def cells(self) -> np.ndarray:
        n = self.R * self.T * self.S
        buf = (ctypes.c_uint8 * (n * 160)).from_address(self._lib.oracle_cells(self._st))
        return np.frombuffer(buf, dtype=CELL_DTYPE).reshape(self.R, self.T, self.S).copy()

    def spans(self) -> np.ndarray:
        self.phase_times()
        n = self.R * self.T * (self.P + 1)
        buf = (ctypes.c_uint8 * (n * 32)).from_address(self._lib.oracle_spans(self._st))
        return np.frombuffer(buf, dtype=SPAN_DTYPE).reshape(self.R, self.T, self.P + 1).copy()

    def record_bytes(self) -> int:
        return int(self._lib.oracle_record_bytes(self._st))

    def records(self) -> np.ndarray:
        """The [R][T] table of fixed-size records (R17) as uint8 [R*T, record_bytes]."""
        out = np.zeros((self.R * self.T, self.record_bytes()), dtype=np.uint8)
        self._lib.oracle_encode_records(self._st, out.ctypes.data)
        return out

    def diagnose(self) -> dict:
        R, T, S, P = self.R, self.T, self.S, self.P
        out = dict(sig_stats=np.zeros((T, S), dtype=STAT_DTYPE),
                   sig_flags=np.zeros((T, S, R), dtype=np.uint8),
                   span_stats=np.zeros((T, P + 1), dtype=STAT_DTYPE),
                   span_flags=np.zeros((T, P + 1, R), dtype=np.uint8),
                   rank_score=np.zeros((T, R), dtype=np.uint32),
                   step_anomalous=np.zeros(T, dtype=np.uint32))
        self._lib.oracle_diagnose(self._st, *[out[k].ctypes.data for k in
                                              ("sig_stats", "sig_flags", "span_stats", "span_flags",
                                               "rank_score", "step_anomalous")])
        return out
