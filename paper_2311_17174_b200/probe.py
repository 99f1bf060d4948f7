"""ctypes binding of include/emri_probe.h (libemri_probe.so): the peak probes bench.py quotes its roofline fractions
against.  Measurement helpers, not part of the boundary of include/emri.h."""
import ctypes as C
import os

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libemri_probe.so")
_lib = None
EXPORTS = ("emri_probe_fp64_peak", "emri_probe_fp64_peak3", "emri_probe_hbm_read")


def load():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} is missing: build it with `python -m paper_2311_17174_b200.build`")
        L = C.CDLL(_LIB_PATH)
        L.emri_probe_fp64_peak.argtypes = [C.POINTER(C.c_double), C.c_void_p]
        L.emri_probe_fp64_peak3.argtypes = [C.POINTER(C.c_double), C.c_void_p]
        L.emri_probe_hbm_read.argtypes = [C.c_int64, C.POINTER(C.c_double), C.c_void_p]
        for n in EXPORTS:
            getattr(L, n).restype = C.c_int
        _lib = L
    return _lib


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _call(fn, *args):
    v = C.c_double()
    rc = fn(*args, C.byref(v), _stream())
    if rc:
        raise RuntimeError(f"probe failed ({rc})")
    return v.value


def fp64_peak():
    """TFLOP/s of a chain-free DFMA kernel with a constant operand on the current device"""
    return _call(load().emri_probe_fp64_peak)


def fp64_peak3():
    """TFLOP/s of DFMAs with three fresh vector-register operands (register-file-bound FP64 rate)"""
    return _call(load().emri_probe_fp64_peak3)


def hbm_read(nbytes=4 << 30):
    """GB/s of a streaming read of `nbytes` of device memory"""
    return _call(load().emri_probe_hbm_read, C.c_int64(int(nbytes)))
