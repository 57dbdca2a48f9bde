"""CPU oracle for the longitudinal tracking hot path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes loader around ``oracle/longtrack_oracle.c`` (read ``longtrack_oracle.h``
first: scope, citations, pins).  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.
It imports nothing from ``paper_1610_05801_b200`` and that package imports nothing
from here.  There is no arithmetic of the method in this file: every number comes out
of the C functions.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import (POINTER, Structure, c_double, c_int, c_size_t, c_ubyte, c_ulonglong,
                    c_void_p)

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_C_FILES = ("longtrack_oracle.c", "next_oracle.c")
_SRC = [os.path.join(_HERE, f) for f in _C_FILES + ("map.inc", "programme.inc", "ramp.inc",
                                                     "longtrack_oracle.h", "next_oracle.h")]
_LIB = os.path.join(_HERE, "liblongtrack_oracle.so")

EULER_CROMER, LEAPFROG, RUTH4 = 0, 1, 2
INTEGRATORS = {"euler_cromer": EULER_CROMER, "leapfrog": LEAPFROG, "ruth4": RUTH4}

# gcc flags: plain two-rounding arithmetic (reading G21: no FMA contraction)
CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra"]


class Params(Structure):
    _fields_ = [("circumference_m", c_double), ("gamma", c_double), ("alpha_c", c_double),
                ("p0c_eV", c_double), ("charge_e", c_double), ("harmonic", c_int),
                ("voltage_V", c_double), ("phi_s", c_double), ("ratio2", c_double),
                ("integrator", c_int)]


class Derived(Structure):
    _fields_ = [(k, c_double) for k in
                ("R", "beta", "eta", "A", "d", "kappa", "K", "z_max", "H_sep")]


class Moments(Structure):
    _fields_ = [("mean_z", c_double), ("rms_z", c_double), ("mean_d", c_double),
                ("rms_d", c_double), ("cov_zd", c_double), ("n_in_bucket", c_ulonglong)]


MOMENTS_DTYPE = np.dtype([("mean_z", "f8"), ("rms_z", "f8"), ("mean_d", "f8"),
                          ("rms_d", "f8"), ("cov_zd", "f8"), ("n_in_bucket", "u8")])


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    newest = max(os.path.getmtime(s) for s in _SRC)
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        cmd = ["gcc", *CFLAGS, "-o", _LIB, *_C_FILES, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = POINTER(c_double)
        pp = POINTER(Params)
        L.lto_derive.argtypes = [pp, POINTER(Derived)]
        L.lto_derive.restype = c_int
        L.lto_kick.argtypes = [pp, c_double]
        L.lto_kick.restype = c_double
        L.lto_one_turn.argtypes = [pp, dp, dp, c_size_t]
        L.lto_one_turn.restype = None
        L.lto_one_turn_ec_adjoint.argtypes = [pp, dp, dp, c_size_t]
        L.lto_one_turn_ec_adjoint.restype = None
        L.lto_track.argtypes = [pp, dp, dp, c_size_t, c_ulonglong]
        L.lto_track.restype = None
        L.lto_track_ld.argtypes = [pp, c_void_p, c_void_p, c_size_t, c_ulonglong]
        L.lto_track_ld.restype = None
        L.lto_track_moments.argtypes = [pp, dp, dp, c_size_t, c_ulonglong, c_void_p]
        L.lto_track_moments.restype = None
        L.lto_moments_of.argtypes = [pp, dp, dp, c_size_t, POINTER(Moments)]
        L.lto_moments_of.restype = None
        L.lto_hamiltonian.argtypes = [pp, c_double, c_double]
        L.lto_hamiltonian.restype = c_double
        L.lto_hamiltonian_n.argtypes = [pp, dp, dp, c_size_t, dp]
        L.lto_hamiltonian_n.restype = None
        L.lto_in_bucket.argtypes = [pp, c_double, c_double]
        L.lto_in_bucket.restype = c_int
        L.lto_bucket_count.argtypes = [pp, dp, dp, c_size_t]
        L.lto_bucket_count.restype = c_ulonglong
        L.lto_bucket_mask.argtypes = [pp, dp, dp, c_size_t, POINTER(c_ubyte)]
        L.lto_bucket_mask.restype = None
        L.lto_num_threads.restype = c_int
        ull = POINTER(c_ulonglong)
        L.lto_track_programme.argtypes = [pp, dp, dp, c_size_t, c_ulonglong, dp, dp]
        L.lto_track_programme.restype = None
        L.lto_track_programme_ld.argtypes = [pp, c_void_p, c_void_p, c_size_t, c_ulonglong, dp, dp]
        L.lto_track_programme_ld.restype = None
        L.lto_track_programme_moments.argtypes = [pp, dp, dp, c_size_t, c_ulonglong, dp, dp, c_void_p]
        L.lto_track_programme_moments.restype = None
        L.lto_track_ramp.argtypes = [pp, dp, dp, c_size_t, c_ulonglong, dp, dp, dp]
        L.lto_track_ramp.restype = None
        L.lto_track_ramp_ld.argtypes = [pp, c_void_p, c_void_p, c_size_t, c_ulonglong, dp, dp, dp]
        L.lto_track_ramp_ld.restype = None
        L.lto_track_ramp_moments.argtypes = [pp, dp, dp, c_size_t, c_ulonglong, dp, dp, dp, c_void_p]
        L.lto_track_ramp_moments.restype = None
        L.lto_ramp_numbers.argtypes = [pp, c_double, dp, dp, dp, dp, dp]
        L.lto_ramp_numbers.restype = None
        L.lto_slice_histogram.argtypes = [dp, c_size_t, c_double, c_double, c_int, ull]
        L.lto_slice_histogram.restype = None
        L.lto_track_slices.argtypes = [pp, dp, dp, c_size_t, c_ulonglong, c_double, c_double,
                                       c_int, ull]
        L.lto_track_slices.restype = None
        L.lto_track_transverse.argtypes = [pp, dp, c_int, dp, dp, dp, dp, dp, dp, c_size_t,
                                           c_ulonglong]
        L.lto_track_transverse.restype = None
        L.lto_set_num_threads.argtypes = [c_int]
        _lib = L
    return _lib


def make_params(ring: dict, integrator="leapfrog", ratio2: float = 0.0,
                phi_s: float | None = None) -> Params:
    """ring: dict with the keys of ``Params`` (see workloads.RING)."""
    integ = INTEGRATORS[integrator] if isinstance(integrator, str) else int(integrator)
    return Params(float(ring["circumference_m"]), float(ring["gamma"]),
                  float(ring["alpha_c"]), float(ring["p0c_eV"]),
                  float(ring.get("charge_e", 1.0)), int(ring["harmonic"]),
                  float(ring["voltage_V"]),
                  float(ring.get("phi_s", 0.0) if phi_s is None else phi_s),
                  float(ratio2), integ)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(POINTER(c_double))


def derive(p: Params) -> dict:
    out = Derived()
    rc = lib().lto_derive(ctypes.byref(p), ctypes.byref(out))
    assert rc == 0
    return {k: getattr(out, k) for k, _ in Derived._fields_}


def kick(p: Params, z: float) -> float:
    return lib().lto_kick(ctypes.byref(p), float(z))


def one_turn(p: Params, z, delta):
    """Returns new (z, delta) arrays after one turn (inputs untouched)."""
    z, zp = _f64(np.array(z, dtype=np.float64, copy=True).ravel())
    d, dp_ = _f64(np.array(delta, dtype=np.float64, copy=True).ravel())
    lib().lto_one_turn(ctypes.byref(p), zp, dp_, z.size)
    return z, d


def one_turn_ec_adjoint(p: Params, z, delta):
    z, zp = _f64(np.array(z, dtype=np.float64, copy=True).ravel())
    d, dp_ = _f64(np.array(delta, dtype=np.float64, copy=True).ravel())
    lib().lto_one_turn_ec_adjoint(ctypes.byref(p), zp, dp_, z.size)
    return z, d


def track(p: Params, z, delta, turns: int):
    """Returns new (z, delta) arrays after ``turns`` turns (inputs untouched)."""
    z, zp = _f64(np.array(z, dtype=np.float64, copy=True).ravel())
    d, dp_ = _f64(np.array(delta, dtype=np.float64, copy=True).ravel())
    lib().lto_track(ctypes.byref(p), zp, dp_, z.size, int(turns))
    return z, d


def track_ld(p: Params, z, delta, turns: int):
    """Same map in 80-bit long double; returns np.longdouble arrays."""
    z = np.ascontiguousarray(np.array(z, dtype=np.longdouble, copy=True).ravel())
    d = np.ascontiguousarray(np.array(delta, dtype=np.longdouble, copy=True).ravel())
    assert z.dtype.itemsize == 16, "expects x86-64 80-bit long double padded to 16 bytes"
    lib().lto_track_ld(ctypes.byref(p), z.ctypes.data, d.ctypes.data, z.size, int(turns))
    return z, d


def track_moments(p: Params, z, delta, turns: int):
    """Returns (z, delta, moments[turns]); moments[t] = state after turn t+1."""
    z, zp = _f64(np.array(z, dtype=np.float64, copy=True).ravel())
    d, dp_ = _f64(np.array(delta, dtype=np.float64, copy=True).ravel())
    out = np.zeros(int(turns), dtype=MOMENTS_DTYPE)
    assert out.dtype.itemsize == ctypes.sizeof(Moments)
    lib().lto_track_moments(ctypes.byref(p), zp, dp_, z.size, int(turns), out.ctypes.data)
    return z, d, out


def moments_of(p: Params, z, delta) -> dict:
    z, zp = _f64(z)
    d, dp_ = _f64(delta)
    out = Moments()
    lib().lto_moments_of(ctypes.byref(p), zp, dp_, z.size, ctypes.byref(out))
    return {k: getattr(out, k) for k, _ in Moments._fields_}


def hamiltonian(p: Params, z, delta):
    z, zp = _f64(np.atleast_1d(z))
    d, dp_ = _f64(np.atleast_1d(delta))
    H = np.empty_like(z)
    lib().lto_hamiltonian_n(ctypes.byref(p), zp, dp_, z.size, H.ctypes.data_as(POINTER(c_double)))
    return H


def bucket_count(p: Params, z, delta) -> int:
    z, zp = _f64(z)
    d, dp_ = _f64(delta)
    return int(lib().lto_bucket_count(ctypes.byref(p), zp, dp_, z.size))


def bucket_mask(p: Params, z, delta):
    z, zp = _f64(z)
    d, dp_ = _f64(delta)
    m = np.empty(z.size, dtype=np.uint8)
    lib().lto_bucket_mask(ctypes.byref(p), zp, dp_, z.size, m.ctypes.data_as(POINTER(c_ubyte)))
    return m.astype(bool)


def num_threads() -> int:
    return int(lib().lto_num_threads())


def set_num_threads(n: int) -> None:
    lib().lto_set_num_threads(int(n))


# ------------------------------------------------------------------ SURVEY.md sec. 8(f) rows f2-f4
def _copy(a):
    return _f64(np.array(a, dtype=np.float64, copy=True).ravel())


def track_programme(p: Params, z, delta, volt_scale, phase_off):
    """f2: one turn per programme entry; returns new (z, delta)."""
    z, zp = _copy(z)
    d, dp_ = _copy(delta)
    a, ap = _f64(volt_scale)
    s, sp = _f64(phase_off)
    assert a.size == s.size
    lib().lto_track_programme(ctypes.byref(p), zp, dp_, z.size, a.size, ap, sp)
    return z, d


def track_programme_ld(p: Params, z, delta, volt_scale, phase_off):
    z = np.ascontiguousarray(np.array(z, dtype=np.longdouble, copy=True).ravel())
    d = np.ascontiguousarray(np.array(delta, dtype=np.longdouble, copy=True).ravel())
    a, ap = _f64(volt_scale)
    s, sp = _f64(phase_off)
    assert a.size == s.size and z.dtype.itemsize == 16
    lib().lto_track_programme_ld(ctypes.byref(p), z.ctypes.data, d.ctypes.data, z.size, a.size,
                                 ap, sp)
    return z, d


def track_programme_moments(p: Params, z, delta, volt_scale, phase_off):
    z, zp = _copy(z)
    d, dp_ = _copy(delta)
    a, ap = _f64(volt_scale)
    s, sp = _f64(phase_off)
    assert a.size == s.size
    out = np.zeros(a.size, dtype=MOMENTS_DTYPE)
    lib().lto_track_programme_moments(ctypes.byref(p), zp, dp_, z.size, a.size, ap, sp,
                                      out.ctypes.data)
    return z, d, out


def _ramp_tables(p0c, volt_scale, phase_off):
    pc, pcp = _f64(p0c)
    turns = pc.size - 1
    assert turns >= 0
    keep = [pc]
    ap = sp = None
    if volt_scale is not None:
        a, ap = _f64(volt_scale)
        assert a.size == turns
        keep.append(a)
    if phase_off is not None:
        s, sp = _f64(phase_off)
        assert s.size == turns
        keep.append(s)
    return turns, pcp, ap, sp, keep


def track_ramp(p: Params, z, delta, p0c, volt_scale=None, phase_off=None):
    """f2 with an energy ramp (G32): p0c has turns+1 entries; returns new (z, delta)."""
    z, zp = _copy(z)
    d, dp_ = _copy(delta)
    turns, pcp, ap, sp, _keep = _ramp_tables(p0c, volt_scale, phase_off)
    lib().lto_track_ramp(ctypes.byref(p), zp, dp_, z.size, turns, pcp, ap, sp)
    return z, d


def track_ramp_ld(p: Params, z, delta, p0c, volt_scale=None, phase_off=None):
    z = np.ascontiguousarray(np.array(z, dtype=np.longdouble, copy=True).ravel())
    d = np.ascontiguousarray(np.array(delta, dtype=np.longdouble, copy=True).ravel())
    assert z.dtype.itemsize == 16
    turns, pcp, ap, sp, _keep = _ramp_tables(p0c, volt_scale, phase_off)
    lib().lto_track_ramp_ld(ctypes.byref(p), z.ctypes.data, d.ctypes.data, z.size, turns, pcp, ap, sp)
    return z, d


def track_ramp_moments(p: Params, z, delta, p0c, volt_scale=None, phase_off=None):
    z, zp = _copy(z)
    d, dp_ = _copy(delta)
    turns, pcp, ap, sp, _keep = _ramp_tables(p0c, volt_scale, phase_off)
    out = np.zeros(turns, dtype=MOMENTS_DTYPE)
    lib().lto_track_ramp_moments(ctypes.byref(p), zp, dp_, z.size, turns, pcp, ap, sp,
                                 out.ctypes.data)
    return z, d, out


def ramp_numbers(p: Params, p0c: float) -> dict:
    """mc2, beta, eta, A, d at reference momentum p0c (G32)."""
    v = [ctypes.c_double() for _ in range(5)]
    lib().lto_ramp_numbers(ctypes.byref(p), float(p0c), *[ctypes.byref(x) for x in v])
    return dict(zip(("mc2", "beta", "eta", "A", "d"), (x.value for x in v)))


def slice_histogram(z, z_lo: float, z_hi: float, n_slices: int):
    """f4: uint64[n_slices + 2] = [below, slices..., above]."""
    z, zp = _f64(z)
    h = np.zeros(n_slices + 2, dtype=np.uint64)
    lib().lto_slice_histogram(zp, z.size, float(z_lo), float(z_hi), int(n_slices),
                              h.ctypes.data_as(POINTER(c_ulonglong)))
    return h


def track_slices(p: Params, z, delta, turns: int, z_lo: float, z_hi: float, n_slices: int):
    z, zp = _copy(z)
    d, dp_ = _copy(delta)
    h = np.zeros((int(turns), n_slices + 2), dtype=np.uint64)
    lib().lto_track_slices(ctypes.byref(p), zp, dp_, z.size, int(turns), float(z_lo),
                           float(z_hi), int(n_slices), h.ctypes.data_as(POINTER(c_ulonglong)))
    return z, d, h


def track_transverse(p: Params, matrices, x, xp, y, yp, z, delta, turns: int):
    """f3: matrices = array [n_seg, 4, 4]; returns new (x, xp, y, yp, z, delta); z/delta may be None."""
    m, mp = _f64(np.asarray(matrices, dtype=np.float64).reshape(-1, 16))
    arrs = [_copy(a) for a in (x, xp, y, yp)]
    n = arrs[0][0].size
    if z is None:
        zz = dd = None
        zp = dp_ = None
    else:
        zz, zp = _copy(z)
        dd, dp_ = _copy(delta)
    lib().lto_track_transverse(ctypes.byref(p), mp, m.shape[0], arrs[0][1], arrs[1][1], arrs[2][1],
                               arrs[3][1], zp, dp_, n, int(turns))
    return tuple(a for a, _ in arrs) + (zz, dd)
