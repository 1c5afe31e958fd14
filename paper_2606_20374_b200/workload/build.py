"""Loaders of the two expander builds (see expand_core.h)."""
import ctypes

from .._build import build_workload_device, build_workload_host


def load_host_lib() -> ctypes.CDLL:
    lib = ctypes.CDLL(build_workload_host())
    lib.wl_expand_host.restype = ctypes.c_int
    lib.wl_expand_host.argtypes = [ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint32,
                                   ctypes.c_void_p, ctypes.c_int]
    lib.wl_perm_host.restype = ctypes.c_uint64
    lib.wl_perm_host.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64]
    lib.wl_desc_bytes.restype = ctypes.c_uint
    return lib


def load_device_lib() -> ctypes.CDLL:
    lib = ctypes.CDLL(build_workload_device())
    lib.wl_expand_device.restype = ctypes.c_int
    lib.wl_expand_device.argtypes = [ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint32,
                                     ctypes.c_void_p, ctypes.c_void_p]
    return lib
