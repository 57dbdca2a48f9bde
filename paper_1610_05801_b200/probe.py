"""ctypes binding of liblongtrack_probe.so (include/longtrack_probe.h) -- argument marshalling only.

The FP64-pipe probes bench.py uses for its roofline denominators.  Measurement tooling: kept in
its own library so that liblongtrack.so exports the tracking calls only.  Importing this module
loads the library and raises ImportError when it is missing; there is no CPU fallback.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_double, c_int, c_longlong

from .longtrack import OK, LongtrackError

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("LONGTRACK_PROBE_LIB") or os.path.join(_HERE, "liblongtrack_probe.so")


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s is missing: build it with `python -m paper_1610_05801_b200.build`" % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    sig = {
        "lt_probe_fp64": (c_int, [c_int, c_int, c_int, c_longlong, POINTER(c_double), POINTER(c_double)]),
        "lt_probe_pipe": (c_int, [c_int, c_int, c_int, c_int, c_longlong, POINTER(c_double),
                                  POINTER(c_double)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    return L, tuple(sig)


_lib, EXPORTS = _load()


def probe_fp64(blocks: int, threads: int, chains: int, iters: int):
    """Returns (FP64 lane-instructions per second, milliseconds) of a dependent-chain DFMA kernel."""
    rate, ms = c_double(), c_double()
    rc = _lib.lt_probe_fp64(blocks, threads, chains, iters, byref(rate), byref(ms))
    if rc != OK:
        raise LongtrackError(rc)
    return rate.value, ms.value


def probe_pipe(kind: int, blocks: int, threads: int, chains: int, iters: int):
    """Returns (FP64 warp-instructions per cycle per sub-partition, SM clock in MHz)."""
    rate, mhz = c_double(), c_double()
    rc = _lib.lt_probe_pipe(kind, blocks, threads, chains, iters, byref(rate), byref(mhz))
    if rc != OK:
        raise LongtrackError(rc)
    return rate.value, mhz.value
