"""Bench hooks (include/flare_probes.h, libflare_probes.so): FP64 DMMA / DFMA issue peaks and an HBM copy measured on
the device, the roofline denominators bench.py reports against.  Not used by the force-field path."""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libflare_probes.so")
EXPORTS = ("flare_probe_fp64_dmma_tflops", "flare_probe_fp64_dfma_tflops", "flare_probe_hbm_copy_gbs")

_lib = None


def load_library():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2204_12573_b200.build`")
        lib = C.CDLL(LIB_PATH)
        lib.flare_probe_fp64_dmma_tflops.argtypes = [C.c_int]
        lib.flare_probe_fp64_dmma_tflops.restype = C.c_double
        lib.flare_probe_fp64_dfma_tflops.argtypes = [C.c_int]
        lib.flare_probe_fp64_dfma_tflops.restype = C.c_double
        lib.flare_probe_hbm_copy_gbs.argtypes = [C.c_int, C.c_size_t]
        lib.flare_probe_hbm_copy_gbs.restype = C.c_double
        _lib = lib
    return _lib


def fp64_dmma_tflops(device: int = 0) -> float:
    return float(load_library().flare_probe_fp64_dmma_tflops(int(device)))


def fp64_dfma_tflops(device: int = 0) -> float:
    return float(load_library().flare_probe_fp64_dfma_tflops(int(device)))


def hbm_copy_gbs(device: int = 0, nbytes: int = 1 << 30) -> float:
    return float(load_library().flare_probe_hbm_copy_gbs(int(device), int(nbytes)))
