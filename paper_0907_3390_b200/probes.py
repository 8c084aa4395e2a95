"""Thin Python binding of include/gamer_probes.h (libgamer_probes.so): the measurement aids of bench.py.  Not part of
the hydro path; the product library does not contain them."""
import ctypes
import os

from .hydro import _ptr

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgamer_probes.so")
_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not found: build it with `python -m paper_0907_3390_b200.build`" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        ci, pd = ctypes.c_int, ctypes.POINTER(ctypes.c_double)
        L.gamer_probe_fp32_peak.restype = ci
        L.gamer_probe_fp32_peak.argtypes = [ci, ctypes.c_void_p, pd, pd, ctypes.c_double]
        L.gamer_probe_issue.restype = ci
        L.gamer_probe_issue.argtypes = [ci, ci, pd]
        L.gamer_probe_last_error.restype = ctypes.c_char_p
        L.gamer_probe_last_error.argtypes = []
        _lib = L
    return _lib


def gamer_probe_last_error():
    return lib().gamer_probe_last_error().decode()


def _check(rc):
    if rc != 0:
        raise RuntimeError("gamer_probes: status %d: %s" % (rc, gamer_probe_last_error()))


def gamer_probe_fp32_peak(repeats, d_sink, sm_mhz=0.0):
    """FMA-only micro-benchmark of the FP32 pipe: returns (TFLOP/s, FMAs per clock per SM)."""
    t, l = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(lib().gamer_probe_fp32_peak(int(repeats), _ptr(d_sink), ctypes.byref(t), ctypes.byref(l), float(sm_mhz)))
    return t.value, l.value


def gamer_probe_issue(what, warps_per_smsp=4):
    """Clocks per 3-register FMA (what = 0) or per warp-march along x, y, z (1, 2, 3); DESIGN.md 7."""
    c = ctypes.c_double(0.0)
    _check(lib().gamer_probe_issue(int(what), int(warps_per_smsp), ctypes.byref(c)))
    return c.value
