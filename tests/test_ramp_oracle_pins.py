"""Pins of the energy-ramp oracle (oracle/ramp.inc; SURVEY.md sec. 8(f) row f2 "gamma ramps per
turn"; reading G32 of DESIGN.md) against what the mathematics fixes.  Nothing here touches the
CUDA path.  Each test is chosen so that a plausible mistake (beta or eta taken at the wrong end
of the turn, the reference's own energy gain dropped or with the wrong sign, delta not re-expressed
relative to the new reference, the Ruth4 momentum steps not summing to the turn's step, the wrong
table index) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_1610_05801_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
INTEGRATORS = ("euler_cromer", "leapfrog", "ruth4")


def P(integrator="leapfrog", ratio2=0.0, **ring_over):
    ring = dict(wl.RING)
    ring.update(ring_over)
    return oracle.make_params(ring, integrator, ratio2)


def golden():
    rows, tab, numbers = [], {}, {}
    for line in open(os.path.join(GOLD, "ramp_values.txt")):
        if line.startswith("# mc2"):
            tok = line[1:].replace("=", " ").split()
            numbers = {tok[i]: float(tok[i + 1]) for i in range(0, len(tok), 2)}
        elif line.startswith("#") and "=" in line:
            k, v = line[1:].split("=")
            tab[k.strip()] = [float(x) for x in v.split()]
        elif not line.startswith("#"):
            rows.append(line.split())
    return rows, tab, numbers


def test_ramp_hand_iterated_values():
    """40-digit hand iteration (tests/golden/ramp_values.txt, mpmath only) over a violent ramp
    (up, down, flat, up) with a voltage and a phase programme: pins which end of the turn
    beta/eta/A/d are taken at, the sign and size of the reference's own gain, the re-scaling
    pb/pa, the Ruth4 intermediate momenta and the table index."""
    rows, tab, _ = golden()
    assert len(rows) == 3 * 2 * 4 * 4
    for name, r, z0, d0, t, z_ref, d_ref in rows:
        t = int(t)
        z, d = oracle.track_ramp(P(name, float(r)), [float(z0)], [float(d0)], tab["p0c"][:t + 1],
                                 tab["volt_scale"][:t], tab["phase_off"][:t])
        z_ref, d_ref = float(z_ref), float(d_ref)
        assert abs(z[0] - z_ref) <= 2e-14 * max(abs(z_ref), 0.1), (name, r, z0, d0, t)
        assert abs(d[0] - d_ref) <= 2e-14 * max(abs(d_ref), 1e-3), (name, r, z0, d0, t)


def test_momentum_dependent_ring_numbers():
    """mc2, A(p), d(p) against the 40-digit line of the golden file; at the create momentum they
    are the constants of the plain map; eta crosses zero at transition gamma = 1/sqrt(alpha_c)."""
    _, _, num = golden()
    p = P()
    at26, at28 = oracle.ramp_numbers(p, 26e9), oracle.ramp_numbers(p, 28e9)
    assert abs(at26["mc2"] / num["mc2"] - 1) <= 4e-16
    assert abs(at26["A"] / num["A(26e9)"] - 1) <= 1e-15 and abs(at26["d"] / num["d(26e9)"] - 1) <= 1e-14
    assert abs(at28["A"] / num["A(28e9)"] - 1) <= 1e-15 and abs(at28["d"] / num["d(28e9)"] - 1) <= 1e-14
    g = oracle.derive(p)
    assert abs(at26["A"] / g["A"] - 1) <= 1e-15 and abs(at26["eta"] / g["eta"] - 1) <= 1e-13
    gamma_t = 1 / math.sqrt(wl.RING["alpha_c"])
    p_t = at26["mc2"] * math.sqrt(gamma_t ** 2 - 1)
    assert abs(oracle.ramp_numbers(p, p_t)["eta"]) <= 1e-17
    assert oracle.ramp_numbers(p, 0.9 * p_t)["eta"] < 0 < oracle.ramp_numbers(p, 1.1 * p_t)["eta"]


@pytest.mark.parametrize("integrator", INTEGRATORS)
@pytest.mark.parametrize("ratio2", [0.0, 0.5])
def test_flat_ramp_is_the_plain_map(integrator, ratio2):
    """p0c constant at the create value: the sub-step reduces to the plain map (the only
    difference is beta computed from p instead of gamma: rounding level)."""
    p = P(integrator, ratio2)
    z0, d0 = wl.gaussian_bunch(300, 0.23, 5, ratio2=ratio2)
    N = 1000
    z, d = oracle.track_ramp(p, z0, d0, np.full(N + 1, wl.RING["p0c_eV"]))
    zt, dt = oracle.track(p, z0, d0, N)
    g = oracle.derive(p)
    assert np.max(np.abs(z - zt)) / g["z_max"] <= 1e-11
    assert np.max(np.abs(d - dt)) / 2e-3 <= 1e-11
    # and with tables: the RF programme map
    a, psi = wl.rf_programme(N, 9)
    z, d = oracle.track_ramp(p, z0, d0, np.full(N + 1, wl.RING["p0c_eV"]), a, psi)
    zt, dt = oracle.track_programme(p, z0, d0, a, psi)
    assert np.max(np.abs(z - zt)) / g["z_max"] <= 1e-10
    assert np.max(np.abs(d - dt)) / 2e-3 <= 1e-10


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_without_rf_the_absolute_momentum_is_conserved(integrator):
    """V = 0: p0 (1 + delta) of every particle is a constant of the motion whatever the ramp
    does (the kick line only re-expresses delta relative to the new reference), and z moves by
    the sum of the drifts with the delta of each sub-step."""
    p = P(integrator)
    rng = np.random.default_rng(8)
    N = 200
    p0c = 26e9 * np.cumprod(np.concatenate([[1.0], 1 + 1e-3 * rng.normal(size=N)]))
    z0, d0 = wl.gaussian_bunch(50, 0.23, 6)
    z, d = oracle.track_ramp(p, z0, d0, p0c, np.zeros(N), np.zeros(N))
    assert np.max(np.abs((1 + d) * p0c[-1] / ((1 + d0) * p0c[0]) - 1)) <= 1e-13
    if integrator == "euler_cromer":                   # closed form of z: full drifts d(pa) delta_after
        zz, P_abs = z0.copy(), (1 + d0) * p0c[0]
        for t in range(N):
            dl = P_abs / p0c[t + 1] - 1
            zz = zz - 2 * oracle.ramp_numbers(p, p0c[t + 1])["d"] * dl
        assert np.max(np.abs(z - zz)) <= 1e-9 * np.max(np.abs(zz - z0))


@pytest.mark.parametrize("integrator", INTEGRATORS)
@pytest.mark.parametrize("ratio2", [0.0, 0.5])
def test_one_turn_jacobian_determinant_is_pb_over_pa(integrator, ratio2):
    """The map is symplectic in (z, delta p); in (z, delta) every turn shrinks the area by
    exactly p0c[t]/p0c[t+1] (adiabatic damping) -- not 1, and not its square."""
    p = P(integrator, ratio2)
    pb, pa = 26e9, 26.8e9
    for z0, d0 in ((0.1, 1e-3), (-0.5, 2e-3), (0.3, -1e-3)):
        ez, ed = 1e-6, 1e-8
        zs = [z0 + ez, z0 - ez, z0, z0]
        ds = [d0, d0, d0 + ed, d0 - ed]
        z, d = oracle.track_ramp_ld(p, zs, ds, [pb, pa], [1.0], [0.4])
        J = np.array([[(z[0] - z[1]) / (2 * ez), (z[2] - z[3]) / (2 * ed)],
                      [(d[0] - d[1]) / (2 * ez), (d[2] - d[3]) / (2 * ed)]], dtype=np.longdouble)
        det = float(J[0, 0] * J[1, 1] - J[0, 1] * J[1, 0])
        assert abs(det - pb / pa) <= 1e-8, (z0, d0, det)
        assert abs(det - 1) > 1e-2 and abs(det - (pb / pa) ** 2) > 1e-2


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_synchronous_particle_stays_on_the_reference(integrator):
    """With psi_t = arcsin(D_t / (pb a_t A(pb))) the RF gives the particle at z = 0, delta = 0
    exactly the reference's gain: it stays at the origin (Ruth4: up to the change of beta within
    a turn, ~1e-9 relative of the gain).  The wrong sign of the gain term, or A taken at the
    wrong end of the turn, moves it by ~1e-5 per turn."""
    p = P(integrator)
    N = 2000
    p0c, a, psi = wl.energy_ramp(N, 26e9, 26.5e9)
    assert np.all(np.diff(p0c) > 0) and 0.1 < psi[N // 2] < 1.2
    z, d = oracle.track_ramp(p, [0.0], [0.0], p0c, a, psi)
    tol = 1e-13 if integrator != "ruth4" else 1e-9
    assert abs(z[0]) <= tol and abs(d[0]) <= tol * 1e-2
    # wrong sign of the phase: it oscillates about the other fixed point, ~2 phi_s/kappa away
    zmax = max(abs(oracle.track_ramp(p, [0.0], [0.0], p0c[:m + 1], a[:m], -psi[:m])[0][0])
               for m in range(N // 2 - 200, N // 2, 20))
    assert zmax > 0.05


def test_adiabatic_damping_of_a_small_bunch():
    """Slow ramp 26 -> 52 GeV/c over 60000 turns on the synchronous phase: the longitudinal
    emittance in (z, delta p) is an adiabatic invariant, so rms_z * rms_delta * p0c is conserved
    (while p0c doubles), and the bunch stays matched: rms_delta / rms_z follows the small-
    amplitude ratio sqrt(A cos(phi_s) kappa / (eta C)) of the energy reached."""
    p = P("leapfrog")
    N = 60_000
    p0c, a, psi = wl.energy_ramp(N, 26e9, 52e9)
    z0, d0 = wl.gaussian_bunch(4000, 0.03, 12)
    z, d = oracle.track_ramp(p, z0, d0, p0c, a, psi)
    e0 = np.std(z0) * np.std(d0) * p0c[0]
    e1 = np.std(z) * np.std(d) * p0c[-1]
    assert abs(e1 / e0 - 1) <= 0.02, e1 / e0
    assert abs(np.std(z) * np.std(d) / (np.std(z0) * np.std(d0)) - 0.5) <= 0.02
    end = oracle.ramp_numbers(p, p0c[-1])
    g = oracle.derive(p)
    ratio = math.sqrt(end["A"] * a[-1] * math.cos(psi[-1]) * g["kappa"] / (2 * end["d"]))
    assert abs(np.std(d) / np.std(z) / ratio - 1) <= 0.03
    assert abs(np.mean(z)) <= 5e-3 and abs(np.mean(d)) <= 5e-5


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_fp64_against_its_80_bit_twin(integrator):
    p = P(integrator, 0.5)
    N = 1000
    p0c, a, psi = wl.energy_ramp(N, 26e9, 26.3e9)
    z0, d0 = wl.gaussian_bunch(300, 0.2, 3, ratio2=0.5)
    z, d = oracle.track_ramp(p, z0, d0, p0c, a, psi)
    zl, dl = oracle.track_ramp_ld(p, z0, d0, p0c, a, psi)
    g = oracle.derive(p)
    assert np.max(np.abs(z - zl.astype(np.float64))) / g["z_max"] <= 1e-10
    assert np.max(np.abs(d - dl.astype(np.float64))) / 2e-3 <= 1e-10


def test_ramp_moments_index_and_null_tables():
    p = P("leapfrog")
    N = 7
    p0c, a, psi = wl.energy_ramp(N, 26e9, 26.001e9)
    z0, d0 = wl.gaussian_bunch(500, 0.23, 4)
    z, d, m = oracle.track_ramp_moments(p, z0, d0, p0c, a, psi)
    for t in (0, 3, 6):
        zt, dt = oracle.track_ramp(p, z0, d0, p0c[:t + 2], a[:t + 1], psi[:t + 1])
        ref = oracle.moments_of(p, zt, dt)
        assert m["mean_z"][t] == ref["mean_z"] and m["rms_d"][t] == ref["rms_d"]
        assert m["n_in_bucket"][t] == ref["n_in_bucket"]
    assert np.array_equal(z, zt) and np.array_equal(d, dt)
    # NULL tables mean a = 1, psi = 0
    za, da = oracle.track_ramp(p, z0, d0, p0c)
    zb, db = oracle.track_ramp(p, z0, d0, p0c, np.ones(N), np.zeros(N))
    assert np.array_equal(za, zb) and np.array_equal(da, db)
