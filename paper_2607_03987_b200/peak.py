"""Measurement support for bench.py, not part of the planning library: builds and loads libpakr_peak.so
(csrc/pakr_peak.cu, csrc/pakr_peak.h) -- the FFMA / FFMA2 / mma.sync microbenchmark whose rates stand beside the
nominal ALU peak in the bench line's roofline."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libpakr_peak.so")
_SRC = [os.path.join(_HERE, "csrc", "pakr_peak.cu"), os.path.join(_HERE, "csrc", "pakr_peak.h")]


class _Fp32Peak(C.Structure):
    _fields_ = [("ffma_lane_ops_per_s", C.c_double), ("ffma2_lane_ops_per_s", C.c_double),
                ("scan_mix_lane_ops_per_s", C.c_double), ("sm_clock_mhz", C.c_double), ("sm_count", C.c_int32),
                ("mma_f16_mac_per_s", C.c_double), ("mma_f16_minfold_mac_per_s", C.c_double)]


def build(force: bool = False) -> str:
    """nvcc -gencode arch=compute_100a,code=sm_100a -> paper_2607_03987_b200/libpakr_peak.so (in-tree)."""
    stale = (not os.path.exists(_SO)) or any(os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if force or stale:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = _SO + f".{os.getpid()}.tmp"
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                               "-Xcompiler", "-fPIC", "-shared", "-o", tmp, _SRC[0]])
        os.replace(tmp, _SO)
    return _SO


_lib = None


def measure_fp32_peak(device: int = 0) -> dict:
    """pakr_measure_fp32_peak: sustained FFMA / FFMA2 / scan-mix lane-ops per second and mma.sync MAC/s of the device."""
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.pakr_measure_fp32_peak.restype = C.c_int
        _lib.pakr_measure_fp32_peak.argtypes = [C.c_int, C.POINTER(_Fp32Peak)]
    out = _Fp32Peak()
    st = _lib.pakr_measure_fp32_peak(device, C.byref(out))
    if st != 0:
        raise RuntimeError(f"pakr_measure_fp32_peak failed with status {st}")
    return {k: getattr(out, k) for k, _ in _Fp32Peak._fields_}
