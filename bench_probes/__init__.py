"""ctypes binding of bench_probes/libspiir_probe.so: FP32 pipe probes used by bench.py (not product code)."""
import ctypes as C

from .build import build as _build

_lib = None


def _l():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
    return _lib


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def fp32_peak_probe(reps=20):
    """(FMA lane-operations per second of a dependency-free FFMA loop, ms per launch)."""
    ms, fma = C.c_double(0), C.c_double(0)
    rc = _l().probe_fp32_peak(C.c_int32(reps), C.byref(ms), C.byref(fma), _stream())
    if rc:
        raise RuntimeError("probe_fp32_peak failed: %d" % rc)
    return fma.value * reps / (ms.value * 1e-3), ms.value / reps


def pipe_probe(mode, reps=5):
    """FP32 lane-operations/s of a register-only copy of a hot inner loop (1 recursion, 2 packed / 3 scalar quadratic form)."""
    ms, ops = C.c_double(0), C.c_double(0)
    rc = _l().probe_pipe(C.c_int32(mode), C.c_int32(reps), C.byref(ms), C.byref(ops), _stream())
    if rc:
        raise RuntimeError("probe_pipe failed: %d" % rc)
    return ops.value * reps / (ms.value * 1e-3)
