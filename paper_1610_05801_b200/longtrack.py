"""ctypes binding of liblongtrack.so -- argument marshalling only.

Same names as include/longtrack.h.  Every step of the hot path runs in the CUDA kernels of
the library; nothing here computes.  PyTorch is used by CALLERS for device memory and streams
(tensors are passed as raw device pointers); this module itself does not import torch.

Importing this module loads the library and raises ImportError when it is missing: there is
no CPU fallback and nothing under oracle/ is ever touched from here.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import (POINTER, Structure, byref, c_char_p, c_double, c_int, c_longlong, c_size_t,
                    c_ulonglong, c_void_p)

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# LONGTRACK_LIB overrides the path (e.g. to try a build with other compile-time knobs)
LIB_PATH = os.environ.get("LONGTRACK_LIB") or os.path.join(_HERE, "liblongtrack.so")

EULER_CROMER, LEAPFROG, RUTH4 = 0, 1, 2
INTEGRATORS = {"euler_cromer": EULER_CROMER, "leapfrog": LEAPFROG, "ruth4": RUTH4}

OK, E_NULL, E_PARAM, E_UNSTABLE, E_ALIGN, E_CUDA, E_NOMEM = 0, -1, -2, -3, -4, -5, -6
E_CAPACITY = -7
STATIC_MAX_PARTICLES = 1 << 24    # lt_moments_now_static

OPT_SPLIT_DRIFTS, OPT_CHUNK_TURNS, OPT_FUSED_ILP, OPT_FUSED_BLOCK = 1, 2, 3, 4
OPT_PER_TURN_GRAPH, OPT_PER_TURN_CTAS_PER_SM, OPT_PER_TURN_REVERSE = 5, 6, 7
OPT_FUSED_MODE, OPT_ITEM_TURNS, OPT_WARPS_PER_SMSP, OPT_FLIP_ON_Q = 8, 9, 10, 11
OPT_RAMP_SCALED = 12
OPT_LATTICE_SOURCE = 13
FUSED_AUTO, FUSED_PLAIN, FUSED_PERSISTENT_STATIC, FUSED_PERSISTENT_DYNAMIC = 0, 1, 2, 3
FUSED_PERSISTENT_WRAP = 4
STAT_KERNEL_LAUNCHES, STAT_LAST_GRID, STAT_LAST_BLOCK, STAT_LAST_ILP, STAT_SM_COUNT = 1, 2, 3, 4, 5
STAT_LAST_MODE, STAT_LAST_ITEM_TURNS = 6, 7


class Params(Structure):
    _fields_ = [("circumference_m", c_double), ("gamma", c_double), ("alpha_c", c_double),
                ("p0c_eV", c_double), ("charge_e", c_double), ("harmonic", c_int),
                ("voltage_V", c_double), ("phi_s", c_double), ("ratio2", c_double),
                ("integrator", c_int)]


class Derived(Structure):
    _fields_ = [(k, c_double) for k in
                ("R", "beta", "eta", "A", "d", "kappa", "K", "mu", "z_max", "H_sep")]


MOMENTS_DTYPE = np.dtype([("mean_z", "f8"), ("rms_z", "f8"), ("mean_d", "f8"), ("rms_d", "f8"),
                          ("cov_zd", "f8"), ("n_in_bucket", "u8")])
SUMS_DTYPE = np.dtype([("n", "f8"), ("sum_z", "f8"), ("sum_zz", "f8"), ("sum_d", "f8"),
                       ("sum_dd", "f8"), ("sum_zd", "f8"), ("n_in_bucket", "f8"), ("pad_", "f8")])


class LongtrackError(RuntimeError):
    def __init__(self, code: int, cuda_error: int = 0):
        self.code = code
        self.cuda_error = cuda_error
        msg = _lib.lt_strerror(code).decode()
        if cuda_error:
            msg += " [cudaError %d]" % cuda_error
        super().__init__("liblongtrack: %s (%d)" % (msg, code))


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "%s is missing: build it with `python -m paper_1610_05801_b200.build` "
            "(there is no CPU fallback)" % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    vp, sz, ull = c_void_p, c_size_t, c_ulonglong
    sig = {
        "lt_create": (c_int, [POINTER(Params), POINTER(vp)]),
        "lt_destroy": (c_int, [vp]),
        "lt_derived": (c_int, [vp, POINTER(Derived)]),
        "lt_set_option": (c_int, [vp, c_int, c_longlong]),
        "lt_get_option": (c_int, [vp, c_int, POINTER(c_longlong)]),
        "lt_get_stat": (c_int, [vp, c_int, POINTER(c_longlong)]),
        "lt_strerror": (c_char_p, [c_int]),
        "lt_last_cuda_error": (c_int, [vp]),
        "lt_version": (c_int, []),
        "lt_track_fused": (c_int, [vp, vp, vp, sz, ull, vp]),
        "lt_track_fused_f32": (c_int, [vp, vp, vp, sz, ull, vp]),
        "lt_track_per_turn": (c_int, [vp, vp, vp, sz, ull, vp, vp, vp]),
        "lt_track_per_turn_f32": (c_int, [vp, vp, vp, sz, ull, vp, vp, vp]),
        "lt_bucket_count": (c_int, [vp, vp, vp, sz, vp, vp]),
        "lt_bucket_count_f32": (c_int, [vp, vp, vp, sz, vp, vp]),
        "lt_moments_now": (c_int, [vp, vp, vp, sz, vp, vp, vp]),
        "lt_moments_now_static": (c_int, [vp, vp, vp, sz, vp, vp, vp]),
        "lt_moments_from_sums": (c_int, [vp, sz, vp]),
        "lt_track_fused_host": (c_int, [vp, vp, vp, sz, ull, POINTER(ull)]),
        "lt_plan_fused": (c_int, [vp, sz, ull, c_int, c_int, POINTER(c_longlong)]),
        "lt_item_schedule": (c_int, [ctypes.c_uint, ctypes.c_uint, c_int, ctypes.c_uint,
                                     POINTER(ctypes.c_uint), POINTER(ctypes.c_uint),
                                     POINTER(ctypes.c_uint)]),
        # SURVEY.md sec. 8(f) rows f2-f4
        "lt_track_programme": (c_int, [vp, vp, vp, sz, ull, vp, vp, vp]),
        "lt_track_programme_per_turn": (c_int, [vp, vp, vp, sz, ull, vp, vp, vp, vp, vp]),
        "lt_track_ramp": (c_int, [vp, vp, vp, sz, ull, vp, vp, vp, vp]),
        "lt_track_ramp_per_turn": (c_int, [vp, vp, vp, sz, ull, vp, vp, vp, vp, vp, vp]),
        "lt_slice_histogram": (c_int, [vp, vp, sz, c_double, c_double, c_int, vp, vp]),
        "lt_track_slices": (c_int, [vp, vp, vp, sz, ull, c_double, c_double, c_int, vp, vp, vp,
                                    vp]),
        "lt_set_transverse": (c_int, [vp, vp, c_int]),
        "lt_track_transverse_fused": (c_int, [vp, vp, vp, vp, vp, vp, vp, sz, ull, vp]),
        "lt_track_transverse_per_turn": (c_int, [vp, vp, vp, vp, vp, vp, vp, sz, ull, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    return L, tuple(sig)


_lib, EXPORTS = _load()


def make_params(ring: dict, integrator="leapfrog", ratio2: float = 0.0,
                phi_s: float | None = None) -> Params:
    integ = INTEGRATORS[integrator] if isinstance(integrator, str) else int(integrator)
    return Params(float(ring["circumference_m"]), float(ring["gamma"]), float(ring["alpha_c"]),
                  float(ring["p0c_eV"]), float(ring.get("charge_e", 1.0)), int(ring["harmonic"]),
                  float(ring["voltage_V"]),
                  float(ring.get("phi_s", 0.0) if phi_s is None else phi_s), float(ratio2), integ)


def _ptr(x) -> int:
    """Raw address of a torch tensor (device or host), a numpy array, an int or None."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    return int(x.ctypes.data)


class Tracker:
    """lt_create / lt_destroy with the track calls as methods (names as in longtrack.h)."""

    def __init__(self, ring: dict, integrator="leapfrog", ratio2: float = 0.0,
                 phi_s: float | None = None):
        self.params = make_params(ring, integrator, ratio2, phi_s)
        self._h = c_void_p()
        rc = _lib.lt_create(byref(self.params), byref(self._h))
        if rc != OK:
            raise LongtrackError(rc)

    def _check(self, rc: int):
        if rc != OK:
            raise LongtrackError(rc, _lib.lt_last_cuda_error(self._h) if rc == E_CUDA else 0)

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:     # _lib is None at interpreter exit
            _lib.lt_destroy(self._h)
            self._h = None

    __del__ = close

    def derived(self) -> dict:
        out = Derived()
        self._check(_lib.lt_derived(self._h, byref(out)))
        return {k: getattr(out, k) for k, _ in Derived._fields_}

    def set_option(self, option: int, value: int):
        self._check(_lib.lt_set_option(self._h, option, int(value)))

    def get_option(self, option: int) -> int:
        v = c_longlong()
        self._check(_lib.lt_get_option(self._h, option, byref(v)))
        return v.value

    def get_stat(self, stat: int) -> int:
        v = c_longlong()
        self._check(_lib.lt_get_stat(self._h, stat, byref(v)))
        return v.value

    def plan_fused(self, n: int, turns: int, sm_count: int = 148, fp32: bool = False) -> dict:
        """Launch shape lt_track_fused would pick (host logic only, no GPU)."""
        plan = (c_longlong * 7)()
        self._check(_lib.lt_plan_fused(self._h, n, turns, sm_count, 1 if fp32 else 0, plan))
        keys = ("dynamic", "warps_per_smsp", "ctas_per_sm", "threads", "item_turns", "flip_on_q",
                "particles_per_lane")
        return dict(zip(keys, (int(v) for v in plan)))

    # ---- device-pointer calls: z, delta are CUDA tensors (or raw addresses); stream = int
    def track_fused(self, z, delta, n: int, turns: int, stream: int = 0):
        self._check(_lib.lt_track_fused(self._h, _ptr(z), _ptr(delta), n, turns, stream))

    def track_fused_f32(self, z, delta, n: int, turns: int, stream: int = 0):
        self._check(_lib.lt_track_fused_f32(self._h, _ptr(z), _ptr(delta), n, turns, stream))

    def track_per_turn(self, z, delta, n: int, turns: int, moments=None, sums=None,
                       stream: int = 0):
        self._check(_lib.lt_track_per_turn(self._h, _ptr(z), _ptr(delta), n, turns,
                                           _ptr(moments), _ptr(sums), stream))

    def track_per_turn_f32(self, z, delta, n: int, turns: int, moments=None, sums=None,
                           stream: int = 0):
        self._check(_lib.lt_track_per_turn_f32(self._h, _ptr(z), _ptr(delta), n, turns,
                                               _ptr(moments), _ptr(sums), stream))

    def bucket_count(self, z, delta, n: int, count, stream: int = 0):
        self._check(_lib.lt_bucket_count(self._h, _ptr(z), _ptr(delta), n, _ptr(count), stream))

    def bucket_count_f32(self, z, delta, n: int, count, stream: int = 0):
        self._check(_lib.lt_bucket_count_f32(self._h, _ptr(z), _ptr(delta), n, _ptr(count),
                                             stream))

    def moments_now(self, z, delta, n: int, moments=None, sums=None, stream: int = 0):
        self._check(_lib.lt_moments_now(self._h, _ptr(z), _ptr(delta), n, _ptr(moments),
                                        _ptr(sums), stream))

    def moments_now_static(self, z, delta, n: int, moments=None, sums=None, stream: int = 0):
        """lt_moments_now without any device allocation, for callers that may not allocate (a
        service whose own pool holds the whole GPU, a monitoring loop that must not stall or fail
        in an allocation, a plug-in barred from the CUDA heap): partial sums go to a fixed 128 KB
        array built into the library.  n <= STATIC_MAX_PARTICLES, else E_CAPACITY.  The array is
        shared by the whole process: calls that overlap on one GPU race.  First call per device
        looks the array up; make it before any stream capture."""
        self._check(_lib.lt_moments_now_static(self._h, _ptr(z), _ptr(delta), n, _ptr(moments),
                                               _ptr(sums), stream))

    # ---- SURVEY.md sec. 8(f) rows f2-f4 (device pointers; tables are device arrays too)
    def track_programme(self, z, delta, n: int, turns: int, volt_scale, phase_off,
                        stream: int = 0):
        self._check(_lib.lt_track_programme(self._h, _ptr(z), _ptr(delta), n, turns,
                                            _ptr(volt_scale), _ptr(phase_off), stream))

    def track_programme_per_turn(self, z, delta, n: int, turns: int, volt_scale, phase_off,
                                 moments=None, sums=None, stream: int = 0):
        self._check(_lib.lt_track_programme_per_turn(self._h, _ptr(z), _ptr(delta), n, turns,
                                                     _ptr(volt_scale), _ptr(phase_off),
                                                     _ptr(moments), _ptr(sums), stream))

    def track_ramp(self, z, delta, n: int, turns: int, p0c, volt_scale=None, phase_off=None,
                   stream: int = 0):
        """Energy ramp (G32): p0c has turns + 1 entries; the two tables may be None."""
        self._check(_lib.lt_track_ramp(self._h, _ptr(z), _ptr(delta), n, turns, _ptr(p0c),
                                       _ptr(volt_scale), _ptr(phase_off), stream))

    def track_ramp_per_turn(self, z, delta, n: int, turns: int, p0c, volt_scale=None,
                            phase_off=None, moments=None, sums=None, stream: int = 0):
        self._check(_lib.lt_track_ramp_per_turn(self._h, _ptr(z), _ptr(delta), n, turns,
                                                _ptr(p0c), _ptr(volt_scale), _ptr(phase_off),
                                                _ptr(moments), _ptr(sums), stream))

    def slice_histogram(self, z, n: int, z_lo: float, z_hi: float, n_slices: int, hist,
                        stream: int = 0):
        self._check(_lib.lt_slice_histogram(self._h, _ptr(z), n, z_lo, z_hi, n_slices,
                                            _ptr(hist), stream))

    def track_slices(self, z, delta, n: int, turns: int, z_lo: float, z_hi: float,
                     n_slices: int, hist, moments=None, sums=None, stream: int = 0):
        self._check(_lib.lt_track_slices(self._h, _ptr(z), _ptr(delta), n, turns, z_lo, z_hi,
                                         n_slices, _ptr(hist), _ptr(moments), _ptr(sums),
                                         stream))

    def set_transverse(self, matrices):
        """matrices: numpy array [n_seg, 4, 4] (row-major) in host memory, or None to clear."""
        if matrices is None:
            self._check(_lib.lt_set_transverse(self._h, None, 0))
            return
        m = np.ascontiguousarray(matrices, dtype=np.float64).reshape(-1, 16)
        self._check(_lib.lt_set_transverse(self._h, m.ctypes.data, m.shape[0]))

    def track_transverse_fused(self, x, xp, y, yp, z, delta, n: int, turns: int,
                               stream: int = 0):
        self._check(_lib.lt_track_transverse_fused(self._h, _ptr(x), _ptr(xp), _ptr(y), _ptr(yp),
                                                   _ptr(z), _ptr(delta), n, turns, stream))

    def track_transverse_per_turn(self, x, xp, y, yp, z, delta, n: int, turns: int,
                                  stream: int = 0):
        self._check(_lib.lt_track_transverse_per_turn(self._h, _ptr(x), _ptr(xp), _ptr(y),
                                                      _ptr(yp), _ptr(z), _ptr(delta), n, turns,
                                                      stream))

    # ---- host-buffer call
    def track_fused_host(self, z_host, delta_host, n: int, turns: int, want_count: bool = False):
        cnt = c_ulonglong(0)
        self._check(_lib.lt_track_fused_host(self._h, _ptr(z_host), _ptr(delta_host), n, turns,
                                             byref(cnt) if want_count else None))
        return cnt.value if want_count else None


def moments_from_sums(sums: np.ndarray) -> np.ndarray:
    sums = np.ascontiguousarray(sums, dtype=SUMS_DTYPE)
    out = np.zeros(sums.shape, dtype=MOMENTS_DTYPE)
    rc = _lib.lt_moments_from_sums(sums.ctypes.data, sums.size, out.ctypes.data)
    if rc != OK:
        raise LongtrackError(rc)
    return out


def item_schedule(turns: int, item_turns: int, taper: bool = True):
    """[(first turn, length)] of every chunk of a launch (host logic only, no GPU)."""
    n, a, b = ctypes.c_uint(), ctypes.c_uint(), ctypes.c_uint()
    rc = _lib.lt_item_schedule(turns, item_turns, 1 if taper else 0, 0, byref(n), None, None)
    if rc != OK:
        raise LongtrackError(rc)
    out = []
    for c in range(n.value):
        rc = _lib.lt_item_schedule(turns, item_turns, 1 if taper else 0, c, byref(n), byref(a), byref(b))
        if rc != OK:
            raise LongtrackError(rc)
        out.append((a.value, b.value))
    return out


def strerror(code: int) -> str:
    return _lib.lt_strerror(code).decode()


def version() -> int:
    return _lib.lt_version()
