"""Thin ctypes binding of libargus.so (include/argus.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for device memory
and streams.  There is no CPU fallback: if the library cannot be built/loaded or no CUDA device is
present, the calls raise."""
from __future__ import annotations

import ctypes
from typing import Optional

import numpy as np

from ._build import build_argus

OK, EINVAL, ECUDA, ESIZE, ESTATE, ENOMEM = 0, -1, -2, -3, -4, -5
FLAG_SORTED = 0x1
TUNE_GRID_CTAS, TUNE_FORCE_PATH = 1, 2
PATH_AUTO, PATH_SEGMENTED, PATH_GLOBAL, PATH_GROUPED = 0, 1, 2, 3

EVENT_DTYPE = np.dtype(
    [("rank", "<u4"), ("step", "<u4"), ("sig", "<u4"), ("stream", "<u2"), ("phase", "<u2"),
     ("start_ns", "<i8"), ("end_ns", "<i8")])
CELL_DTYPE = np.dtype([("count", "<u8"), ("sum", "<u8"), ("min", "<u8"), ("max", "<u8"),
                       ("hist", "<u4", (32,))])
SPAN_DTYPE = np.dtype([("min_start", "<i8"), ("max_end", "<i8"), ("span", "<u8"), ("n", "<u8")])
STAT_DTYPE = np.dtype([("median", "<u8"), ("mad", "<u8"), ("n_high", "<u4"), ("n_low", "<u4"),
                       ("reserved", "<u8")])
HEADER_DTYPE = np.dtype([("magic", "<u4"), ("version", "<u2"), ("n_phases", "<u2"),
                         ("n_sigs", "<u4"), ("rank", "<u4"), ("step", "<u4"), ("reserved0", "<u4"),
                         ("n_events", "<u8"), ("min_start", "<i8"), ("max_end", "<i8"),
                         ("iter_ns", "<u8"), ("reserved1", "<u8")])

CLUSTER_DTYPE = np.dtype([("count", "<u4"), ("p50_bin", "<u2"), ("p99_bin", "<u2")])
L3_STAT_DTYPE = np.dtype([("q1", "<f8"), ("q3", "<f8"), ("fence", "<f8"), ("x_lo", "<f8"), ("x_hi", "<f8")])
L2_GROUP_DTYPE = np.dtype([("n", "<u4"), ("cls", "<u4"), ("mu", "<f8"), ("sigma", "<f8"), ("cv", "<f8")])
L1_MAX_INTERVALS = 8
L1_INTERVAL_DTYPE = np.dtype([("first", "<u4"), ("last", "<u4"), ("width", "<u4"), ("reserved", "<u4"),
                              ("baseline", "<f8")])
L1_OUT_DTYPE = np.dtype([("cls", "<u4"), ("n_intervals", "<u4"), ("cp_found", "<u4"), ("cp_step", "<u4"),
                         ("cp_ratio", "<f8"), ("interval", L1_INTERVAL_DTYPE, (L1_MAX_INTERVALS,))])

EXPORTS = ["argus_create", "argus_destroy", "argus_record_bytes", "argus_table_bytes",
           "argus_workspace_bytes", "argus_reset", "argus_ingest", "argus_aggregate",
           "argus_aggregate_host", "argus_phase_times", "argus_diagnose", "argus_forget", "argus_pack_planes",
           "argus_diagnose_planes", "argus_diagnose_planes_static", "argus_fine_hist", "argus_kde_clusters", "argus_kde_clusters_records",
           "argus_sparse_bound", "argus_sparse_encode", "argus_triple_bound", "argus_triple_encode",
           "argus_clusters_to_l3", "argus_l3_detect", "argus_l2_groups", "argus_l1_detect", "argus_stats", "argus_refused_count", "argus_l3_path_count",
           "argus_launch_count", "argus_tune", "argus_strerror", "argus_last_cuda_error",
           "argus_version"]


class ArgusConfig(ctypes.Structure):
    _fields_ = [("n_ranks", ctypes.c_uint32), ("n_steps", ctypes.c_uint32),
                ("n_sigs", ctypes.c_uint32), ("n_phases", ctypes.c_uint32),
                ("step_base", ctypes.c_uint32), ("flags", ctypes.c_uint32),
                ("device", ctypes.c_int32), ("max_ungrouped_events", ctypes.c_uint32),
                ("max_spill_events", ctypes.c_uint32), ("reserved", ctypes.c_uint32)]


class ArgusDiagOut(ctypes.Structure):
    _fields_ = [("sig_stats", ctypes.c_void_p), ("sig_flags", ctypes.c_void_p),
                ("span_stats", ctypes.c_void_p), ("span_flags", ctypes.c_void_p),
                ("rank_score", ctypes.c_void_p), ("step_anomalous", ctypes.c_void_p)]


class ArgusPlanes(ctypes.Structure):
    _fields_ = [("sig_sums", ctypes.c_void_p), ("span_ns", ctypes.c_void_p),
                ("n_ranks", ctypes.c_uint32), ("rank_stride", ctypes.c_uint32),
                ("n_sigs", ctypes.c_uint32), ("reserved", ctypes.c_uint32)]


class ArgusKdeParams(ctypes.Structure):
    _fields_ = [("per_octave", ctypes.c_uint32), ("n_bins", ctypes.c_uint32), ("min_count", ctypes.c_uint32),
                ("min_gap_bins", ctypes.c_uint32), ("max_clusters", ctypes.c_uint32), ("reserved", ctypes.c_uint32),
                ("min_frac", ctypes.c_double)]


class ArgusL3In(ctypes.Structure):
    _fields_ = [("count", ctypes.c_void_p), ("p50", ctypes.c_void_p), ("p99", ctypes.c_void_p),
                ("n_keys", ctypes.c_uint32), ("n_ranks", ctypes.c_uint32), ("max_clusters", ctypes.c_uint32),
                ("reserved", ctypes.c_uint32)]


class ArgusL3Params(ctypes.Structure):
    _fields_ = [("n_grid", ctypes.c_uint32), ("reserved", ctypes.c_uint32), ("alpha", ctypes.c_double)]


class ArgusL1Params(ctypes.Structure):
    _fields_ = [("window", ctypes.c_uint32), ("min_seg", ctypes.c_uint32), ("theta", ctypes.c_double),
                ("beta", ctypes.c_double), ("ratio_min", ctypes.c_double), ("rsd_max", ctypes.c_double)]


class ArgusError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"argus error {code}: {msg}")
        self.code = code


_lib = None


def load() -> ctypes.CDLL:
    """Build (if stale) and load libargus.so; declare the prototypes of include/argus.h."""
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build_argus())
    vp, u64, i32 = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int
    cfgp = ctypes.POINTER(ArgusConfig)
    lib.argus_create.restype = i32
    lib.argus_create.argtypes = [cfgp, vp, ctypes.c_size_t, ctypes.POINTER(vp)]
    lib.argus_workspace_bytes.restype = ctypes.c_size_t
    lib.argus_workspace_bytes.argtypes = [cfgp]
    lib.argus_destroy.restype = i32
    lib.argus_destroy.argtypes = [vp]
    lib.argus_record_bytes.restype = ctypes.c_size_t
    lib.argus_record_bytes.argtypes = [cfgp]
    lib.argus_table_bytes.restype = ctypes.c_size_t
    lib.argus_table_bytes.argtypes = [cfgp]
    lib.argus_reset.restype = i32
    lib.argus_reset.argtypes = [vp, vp, vp]
    lib.argus_ingest.restype = i32
    lib.argus_ingest.argtypes = [vp, vp, u64, vp, vp]
    lib.argus_aggregate.restype = i32
    lib.argus_aggregate.argtypes = [vp, vp, u64, vp, vp]
    lib.argus_aggregate_host.restype = i32
    lib.argus_aggregate_host.argtypes = [vp, vp, u64, u64, vp, ctypes.c_uint32, vp, vp]
    lib.argus_phase_times.restype = i32
    lib.argus_phase_times.argtypes = [vp, vp, vp, vp]
    lib.argus_diagnose.restype = i32
    lib.argus_diagnose.argtypes = [vp, vp, ctypes.POINTER(ArgusDiagOut), vp]
    lib.argus_forget.restype = i32
    lib.argus_forget.argtypes = [vp]
    lib.argus_pack_planes.restype = i32
    lib.argus_pack_planes.argtypes = [vp, vp, ctypes.c_uint32, ctypes.c_uint32, vp, vp, ctypes.c_uint32,
                                      ctypes.c_uint32, vp]
    lib.argus_diagnose_planes.restype = i32
    lib.argus_diagnose_planes.argtypes = [vp, ctypes.POINTER(ArgusPlanes), ctypes.POINTER(ArgusDiagOut), vp]
    lib.argus_diagnose_planes_static.restype = i32
    lib.argus_diagnose_planes_static.argtypes = [ctypes.POINTER(ArgusPlanes), ctypes.c_uint32, ctypes.c_uint32,
                                                 ctypes.POINTER(ArgusDiagOut), vp]
    lib.argus_fine_hist.restype = i32
    lib.argus_fine_hist.argtypes = [vp, vp, u64, vp, vp]
    lib.argus_kde_clusters.restype = i32
    lib.argus_kde_clusters.argtypes = [vp, vp, u64, ctypes.POINTER(ArgusKdeParams), vp, vp, vp, vp]
    lib.argus_kde_clusters_records.restype = i32
    lib.argus_kde_clusters_records.argtypes = [vp, vp, ctypes.POINTER(ArgusKdeParams), vp, vp, vp]
    lib.argus_sparse_bound.restype = ctypes.c_size_t
    lib.argus_sparse_bound.argtypes = [ctypes.POINTER(ArgusConfig)]
    lib.argus_triple_bound.restype = ctypes.c_size_t
    lib.argus_triple_bound.argtypes = [ctypes.POINTER(ArgusConfig), ctypes.c_uint32]
    lib.argus_sparse_encode.restype = i32
    lib.argus_sparse_encode.argtypes = [vp, vp, vp, u64, vp, vp]
    lib.argus_triple_encode.restype = i32
    lib.argus_triple_encode.argtypes = [vp, vp, vp, vp, ctypes.c_uint32, vp, u64, vp, vp]
    lib.argus_clusters_to_l3.restype = i32
    lib.argus_clusters_to_l3.argtypes = [vp, vp, ctypes.c_uint32, ctypes.c_uint32, vp, vp, vp, vp]
    lib.argus_l3_detect.restype = i32
    lib.argus_l3_detect.argtypes = [vp, ctypes.POINTER(ArgusL3In), ctypes.POINTER(ArgusL3Params), vp, vp, vp, vp]
    lib.argus_l2_groups.restype = i32
    lib.argus_l2_groups.argtypes = [vp, vp, vp, ctypes.c_uint32, vp, ctypes.c_double, vp, vp, vp, vp, vp]
    lib.argus_l1_detect.restype = i32
    lib.argus_l1_detect.argtypes = [vp, vp, u64, u64, ctypes.c_uint32, ctypes.c_uint32,
                                    ctypes.POINTER(ArgusL1Params), vp, vp]
    lib.argus_stats.restype = i32
    lib.argus_stats.argtypes = [vp, ctypes.POINTER(u64), ctypes.POINTER(u64)]
    lib.argus_refused_count.restype = i32
    lib.argus_refused_count.argtypes = [vp, ctypes.POINTER(u64), ctypes.POINTER(u64)]
    lib.argus_l3_path_count.restype = i32
    lib.argus_l3_path_count.argtypes = [vp, ctypes.POINTER(u64), ctypes.POINTER(u64), ctypes.POINTER(u64)]
    lib.argus_launch_count.restype = i32
    lib.argus_launch_count.argtypes = [vp, ctypes.POINTER(u64), ctypes.POINTER(u64)]
    lib.argus_tune.restype = i32
    lib.argus_tune.argtypes = [vp, i32, ctypes.c_int64]
    lib.argus_strerror.restype = ctypes.c_char_p
    lib.argus_strerror.argtypes = [i32]
    lib.argus_last_cuda_error.restype = i32
    lib.argus_last_cuda_error.argtypes = [vp]
    lib.argus_version.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _ptr(x) -> Optional[int]:
    """Raw address of a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    raise TypeError(type(x))


def _stream(s) -> Optional[int]:
    if s is None:
        import torch
        return torch.cuda.current_stream().cuda_stream or None
    if isinstance(s, int):
        return s or None
    return s.cuda_stream or None


STATIC_MAX_SERIES = 262144


def diagnose_planes_static(d_sig_plane, d_span_plane, n_ranks: int, rank_stride: int, n_sigs: int, n_steps: int,
                           n_phases: int, outs: dict, stream=None) -> None:
    """argus_diagnose_planes_static: the cross-rank rule on planes with no context and no device allocation,
    for a monitor that shares a process with a training job whose allocator already owns the HBM (a cudaMalloc
    from the side may fail, and stalls the device when it does not).  The only scratch, a mark byte per series,
    is a fixed 256 KiB array inside libargus.so, so n_steps * (n_sigs + n_phases + 1) <= STATIC_MAX_SERIES
    (ArgusError ESIZE beyond).  Runs on the current device; the array is shared by all calls on that device, so
    calls that could overlap on the GPU must be ordered by the caller."""
    lib = load()
    pl = ArgusPlanes(_ptr(d_sig_plane), _ptr(d_span_plane), n_ranks, rank_stride, n_sigs, 0)
    o = ArgusDiagOut(*[_ptr(outs.get(k)) for k in ("sig_stats", "sig_flags", "span_stats",
                                                   "span_flags", "rank_score", "step_anomalous")])
    rc = lib.argus_diagnose_planes_static(ctypes.byref(pl), n_steps, n_phases, ctypes.byref(o), _stream(stream))
    if rc != OK:
        raise ArgusError(rc, lib.argus_strerror(rc).decode())


class Argus:
    """One context = one table geometry (R ranks x T steps x S sigs, P phases).  Methods carry the
    names of the C entry points; all work is queued on CUDA streams."""

    def __init__(self, n_ranks: int, n_steps: int, n_sigs: int, n_phases: int, step_base: int = 0,
                 sorted_hint: bool = True, device: int = 0, max_ungrouped_events: int = 0,
                 max_spill_events: int = 0, workspace="torch"):
        """workspace: "torch" = a caller-owned torch uint8 tensor of argus_workspace_bytes (kept in
        self.workspace); None = the library allocates it itself in argus_create; or a tensor."""
        self.lib = load()
        self.cfg = ArgusConfig(n_ranks, n_steps, n_sigs, n_phases, step_base,
                               FLAG_SORTED if sorted_hint else 0, device, max_ungrouped_events,
                               max_spill_events, 0)
        self.R, self.T, self.S, self.P = n_ranks, n_steps, n_sigs, n_phases
        self.device = device
        self.workspace = None
        self._h = None
        if isinstance(workspace, str):
            if workspace != "torch":
                raise ValueError(workspace)
            import torch
            nbytes = self.workspace_bytes
            if nbytes:          # 0: invalid config or no device; argus_create reports which
                workspace = torch.empty(nbytes, dtype=torch.uint8, device=f"cuda:{device}")
            else:
                workspace = None
        self.workspace = workspace
        h = ctypes.c_void_p()
        rc = self.lib.argus_create(ctypes.byref(self.cfg), _ptr(workspace),
                                   0 if workspace is None else workspace.numel(), ctypes.byref(h))
        self._h = h if rc == OK else None
        self._check(rc)

    # ---- plumbing ---------------------------------------------------------------------------
    def _check(self, rc: int) -> None:
        if rc != OK:
            msg = self.lib.argus_strerror(rc).decode()
            if rc == ECUDA and self._h:
                msg += f" [cudaError {self.lib.argus_last_cuda_error(self._h)}]"
            raise ArgusError(rc, msg)

    def close(self) -> None:
        if getattr(self, "_h", None):
            self.lib.argus_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def record_bytes(self) -> int:
        return int(self.lib.argus_record_bytes(ctypes.byref(self.cfg)))

    @property
    def table_bytes(self) -> int:
        return int(self.lib.argus_table_bytes(ctypes.byref(self.cfg)))

    @property
    def workspace_bytes(self) -> int:
        return int(self.lib.argus_workspace_bytes(ctypes.byref(self.cfg)))

    def alloc_records(self):
        import torch
        return torch.empty(self.table_bytes, dtype=torch.uint8, device=f"cuda:{self.device}")

    def alloc_diag(self) -> dict:
        import torch
        dev = f"cuda:{self.device}"
        R, T, S, P = self.R, self.T, self.S, self.P
        u8 = torch.uint8
        return dict(sig_stats=torch.empty(T * S * 32, dtype=u8, device=dev),
                    sig_flags=torch.empty(T * S * R, dtype=u8, device=dev),
                    span_stats=torch.empty(T * (P + 1) * 32, dtype=u8, device=dev),
                    span_flags=torch.empty(T * (P + 1) * R, dtype=u8, device=dev),
                    rank_score=torch.empty(T * R, dtype=torch.int32, device=dev),
                    step_anomalous=torch.empty(T, dtype=torch.int32, device=dev))

    # ---- the C entry points -----------------------------------------------------------------
    def reset(self, d_records, stream=None) -> None:
        self._check(self.lib.argus_reset(self._h, _ptr(d_records), _stream(stream)))

    def ingest(self, h_src, n: int, d_dst, copy_stream) -> None:
        self._check(self.lib.argus_ingest(self._h, _ptr(h_src), n, _ptr(d_dst), _stream(copy_stream)))

    def aggregate(self, d_events, n: int, d_records, stream=None) -> None:
        self._check(self.lib.argus_aggregate(self._h, _ptr(d_events), n, _ptr(d_records),
                                             _stream(stream)))

    def aggregate_host(self, h_events, n: int, chunk_events: int, d_ring, ring_slots: int,
                       d_records, stream=None) -> None:
        self._check(self.lib.argus_aggregate_host(self._h, _ptr(h_events), n, chunk_events,
                                                  _ptr(d_ring), ring_slots, _ptr(d_records),
                                                  _stream(stream)))

    def phase_times(self, d_records, d_spans_out=None, stream=None) -> None:
        self._check(self.lib.argus_phase_times(self._h, _ptr(d_records), _ptr(d_spans_out),
                                               _stream(stream)))

    def diagnose(self, d_records, outs: dict, stream=None) -> None:
        o = ArgusDiagOut(*[_ptr(outs.get(k)) for k in ("sig_stats", "sig_flags", "span_stats",
                                                       "span_flags", "rank_score", "step_anomalous")])
        self._check(self.lib.argus_diagnose(self._h, _ptr(d_records), ctypes.byref(o),
                                            _stream(stream)))

    def forget(self) -> None:
        self._check(self.lib.argus_forget(self._h))

    def pack_planes(self, d_records, sig_lo: int, sig_hi: int, d_sig_plane, d_span_plane,
                    rank_stride: int, rank_offset: int, stream=None) -> None:
        self._check(self.lib.argus_pack_planes(self._h, _ptr(d_records), sig_lo, sig_hi, _ptr(d_sig_plane),
                                               _ptr(d_span_plane), rank_stride, rank_offset, _stream(stream)))

    def diagnose_planes(self, d_sig_plane, d_span_plane, n_ranks: int, rank_stride: int, n_sigs: int,
                        outs: dict, stream=None) -> None:
        pl = ArgusPlanes(_ptr(d_sig_plane), _ptr(d_span_plane), n_ranks, rank_stride, n_sigs, 0)
        o = ArgusDiagOut(*[_ptr(outs.get(k)) for k in ("sig_stats", "sig_flags", "span_stats",
                                                       "span_flags", "rank_score", "step_anomalous")])
        self._check(self.lib.argus_diagnose_planes(self._h, ctypes.byref(pl), ctypes.byref(o),
                                                   _stream(stream)))

    # ---- the paper-literal float algorithms (NEXT-1..3): marshalling only ---------------------------------
    def fine_hist(self, d_events, n: int, d_hist, stream=None) -> None:
        self._check(self.lib.argus_fine_hist(self._h, _ptr(d_events), n, _ptr(d_hist), _stream(stream)))

    @staticmethod
    def kde_params(per_octave: int = 8, n_bins: int = 256, min_count: int = 8, min_gap_bins: Optional[int] = None,
                   max_clusters: int = 8, min_frac: float = 0.02) -> "ArgusKdeParams":
        gap = per_octave // 2 if min_gap_bins is None else min_gap_bins
        return ArgusKdeParams(per_octave, n_bins, min_count, gap, max_clusters, 0, min_frac)

    def kde_clusters(self, d_hist, n_cells: int, params, d_clusters, d_n_clusters, d_density=None, stream=None) -> None:
        self._check(self.lib.argus_kde_clusters(self._h, _ptr(d_hist), n_cells, ctypes.byref(params), _ptr(d_clusters),
                                                _ptr(d_n_clusters), _ptr(d_density), _stream(stream)))

    def kde_clusters_records(self, d_records, params, d_clusters, d_n_clusters, stream=None) -> None:
        self._check(self.lib.argus_kde_clusters_records(self._h, _ptr(d_records), ctypes.byref(params),
                                                        _ptr(d_clusters), _ptr(d_n_clusters), _stream(stream)))

    def sparse_bound(self) -> int:
        return int(self.lib.argus_sparse_bound(ctypes.byref(self.cfg)))

    def triple_bound(self, max_clusters: int) -> int:
        return int(self.lib.argus_triple_bound(ctypes.byref(self.cfg), max_clusters))

    def sparse_encode(self, d_records, d_out, d_offsets, stream=None) -> None:
        self._check(self.lib.argus_sparse_encode(self._h, _ptr(d_records), _ptr(d_out), d_out.numel() * d_out.element_size(),
                                                 _ptr(d_offsets), _stream(stream)))

    def triple_encode(self, d_records, d_clusters, d_n_clusters, max_clusters: int, d_out, d_offsets, stream=None) -> None:
        self._check(self.lib.argus_triple_encode(self._h, _ptr(d_records), _ptr(d_clusters), _ptr(d_n_clusters), max_clusters,
                                                 _ptr(d_out), d_out.numel() * d_out.element_size(), _ptr(d_offsets),
                                                 _stream(stream)))

    def clusters_to_l3(self, d_clusters, max_clusters: int, per_octave: int, d_count, d_p50, d_p99, stream=None) -> None:
        self._check(self.lib.argus_clusters_to_l3(self._h, _ptr(d_clusters), max_clusters, per_octave, _ptr(d_count),
                                                  _ptr(d_p50), _ptr(d_p99), _stream(stream)))

    def l3_detect(self, d_count, d_p50, d_p99, n_keys: int, n_ranks: int, max_clusters: int, d_score, d_stat,
                  d_flags, n_grid: int = 256, alpha: float = 1.5, stream=None) -> None:
        i = ArgusL3In(_ptr(d_count), _ptr(d_p50), _ptr(d_p99), n_keys, n_ranks, max_clusters, 0)
        q = ArgusL3Params(n_grid, 0, alpha)
        self._check(self.lib.argus_l3_detect(self._h, ctypes.byref(i), ctypes.byref(q), _ptr(d_score), _ptr(d_stat),
                                             _ptr(d_flags), _stream(stream)))

    def l2_groups(self, d_records, d_route, d_group_id, z_threshold: float, d_groups, d_z, d_flags, d_xbar,
                  stream=None, n_dims: Optional[int] = None) -> None:
        """d_group_id: [n_dims][R] u32; n_dims defaults to its size / R (a torch tensor or numpy array)."""
        if n_dims is None:
            n_dims = (d_group_id.numel() if hasattr(d_group_id, "numel") else d_group_id.size) // self.R
        self._check(self.lib.argus_l2_groups(self._h, _ptr(d_records), _ptr(d_route), n_dims, _ptr(d_group_id), z_threshold,
                                             _ptr(d_groups), _ptr(d_z), _ptr(d_flags), _ptr(d_xbar), _stream(stream)))

    def l1_detect(self, d_base, series_stride: int, step_stride: int, n_series: int, n_steps: int, d_out,
                  window: int = 8, min_seg: int = 4, theta: float = 1.5, beta: float = 1.25, ratio_min: float = 1.1,
                  rsd_max: float = 0.05, stream=None) -> None:
        q = ArgusL1Params(window, min_seg, theta, beta, ratio_min, rsd_max)
        self._check(self.lib.argus_l1_detect(self._h, _ptr(d_base), series_stride, step_stride, n_series, n_steps,
                                             ctypes.byref(q), _ptr(d_out), _stream(stream)))

    def l3_path_count(self):
        """(keys on the class path, keys on the general path, keys without clusters) since reset."""
        a, b, c = ctypes.c_uint64(), ctypes.c_uint64(), ctypes.c_uint64()
        self._check(self.lib.argus_l3_path_count(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)))
        return a.value, b.value, c.value

    def stats(self):
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        self._check(self.lib.argus_stats(self._h, ctypes.byref(a), ctypes.byref(b)))
        return int(a.value), int(b.value)

    def refused_count(self):
        """(re-queued through the spill area, taken by the overflow list / L2 atomics)"""
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        self._check(self.lib.argus_refused_count(self._h, ctypes.byref(a), ctypes.byref(b)))
        return int(a.value), int(b.value)

    def launch_count(self):
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        self._check(self.lib.argus_launch_count(self._h, ctypes.byref(a), ctypes.byref(b)))
        return int(a.value), int(b.value)

    def tune(self, which: int, value: int) -> None:
        self._check(self.lib.argus_tune(self._h, which, value))

    # ---- host-side views of device results (test / report convenience; no arithmetic) ---------
    def records_to_host(self, d_records) -> np.ndarray:
        return d_records.cpu().numpy().reshape(self.R * self.T, self.record_bytes)

    def split_records(self, rec: np.ndarray):
        """uint8 [R*T, record_bytes] -> (headers [R,T], spans [R,T,P+1], cells [R,T,S])."""
        R, T, S, P = self.R, self.T, self.S, self.P
        hdr = rec[:, :64].copy().view(HEADER_DTYPE).reshape(R, T)
        sp = rec[:, 64:64 + 32 * (P + 1)].copy().view(SPAN_DTYPE).reshape(R, T, P + 1)
        ce = rec[:, 64 + 32 * (P + 1):].copy().view(CELL_DTYPE).reshape(R, T, S)
        return hdr, sp, ce

    def diag_to_host(self, outs: dict) -> dict:
        R, T, S, P = self.R, self.T, self.S, self.P
        return dict(
            sig_stats=outs["sig_stats"].cpu().numpy().view(STAT_DTYPE).reshape(T, S),
            sig_flags=outs["sig_flags"].cpu().numpy().reshape(T, S, R),
            span_stats=outs["span_stats"].cpu().numpy().view(STAT_DTYPE).reshape(T, P + 1),
            span_flags=outs["span_flags"].cpu().numpy().reshape(T, P + 1, R),
            rank_score=outs["rank_score"].cpu().numpy().view(np.uint32).reshape(T, R),
            step_anomalous=outs["step_anomalous"].cpu().numpy().view(np.uint32).reshape(T))
