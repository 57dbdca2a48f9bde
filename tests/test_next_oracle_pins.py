"""Pins of the oracle functions for SURVEY.md sec. 8(f) rows f2 (RF programme), f3 (transverse
linear maps) and f4 (slicing) against what the mathematics fixes.  None of these tests touches
the CUDA path; each is chosen so that a plausible mistake in oracle/next_oracle.c or
oracle/programme.inc (wrong table index, dropped offset, transposed matrix, wrong segment order,
off-by-one slice, wrong edge rule) fails at least one of them.
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


def small_bunch(n=200, seed=3, sigma_z=0.23):
    return wl.gaussian_bunch(n, sigma_z, seed)


# ================================================================== f2: RF programme
def programme_rows(name="programme_values.txt"):
    rows, a, psi = [], None, None
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("# volt_scale"):
            a = [float(x) for x in line.split("=")[1].split()]
        elif line.startswith("# phase_off"):
            psi = [float(x) for x in line.split("=")[1].split()]
        elif not line.startswith("#"):
            rows.append(line.split())
    return rows, a, psi


def test_programme_hand_iterated_values():
    """40-digit hand iteration (tests/golden/programme_values.txt, mpmath only): pins the
    table index (entry t <-> turn t+1), the sign and place of psi, the 2 psi of the second
    harmonic and that all three Ruth4 sub-kicks use the same entry."""
    rows, a, psi = programme_rows()
    assert len(rows) == 3 * 2 * 4 * 4
    for name, r, z0, d0, t, z_ref, d_ref in rows:
        t = int(t)
        z, d = oracle.track_programme(P(name, float(r)), [float(z0)], [float(d0)], a[:t], psi[:t])
        z_ref, d_ref = float(z_ref), float(d_ref)
        assert abs(z[0] - z_ref) <= 1e-14 * max(abs(z_ref), 0.1), (name, r, z0, d0, t)
        assert abs(d[0] - d_ref) <= 1e-14 * max(abs(d_ref), 1e-3), (name, r, z0, d0, t)


def test_programme_hand_iterated_values_with_synchronous_phase():
    """The same programme at phi_s = 0.3 and -0.7, r = 0 and 0.25
    (tests/golden/programme_phi_s_values.txt, mpmath only): pins the phi_s branch of
    programme.inc -- sign of phi_s, sin(phi_s) subtracted unshifted by psi_t but scaled by a_t,
    no phi_s in the 2h term (G3, G28)."""
    rows, a, psi = programme_rows("programme_phi_s_values.txt")
    assert len(rows) == 3 * 2 * 2 * 4 * 4
    for name, phi, r, z0, d0, t, z_ref, d_ref in rows:
        t = int(t)
        p = oracle.make_params(wl.RING, name, float(r), phi_s=float(phi))
        z, d = oracle.track_programme(p, [float(z0)], [float(d0)], a[:t], psi[:t])
        z_ref, d_ref = float(z_ref), float(d_ref)
        assert abs(z[0] - z_ref) <= 1e-14 * max(abs(z_ref), 0.1), (name, phi, r, z0, d0, t)
        assert abs(d[0] - d_ref) <= 1e-14 * max(abs(d_ref), 1e-3), (name, phi, r, z0, d0, t)


@pytest.mark.parametrize("integrator", INTEGRATORS)
@pytest.mark.parametrize("ratio2", [0.0, 0.5])
def test_trivial_programme_returns_the_bits_of_the_plain_map(integrator, ratio2):
    p = P(integrator, ratio2)
    z0, d0 = small_bunch()
    za, da = oracle.track(p, z0, d0, 300)
    zb, db = oracle.track_programme(p, z0, d0, np.ones(300), np.zeros(300))
    assert np.array_equal(za, zb) and np.array_equal(da, db)


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_constant_voltage_scale_equals_a_ring_with_that_voltage(integrator):
    z0, d0 = small_bunch()
    a = 0.6
    za, da = oracle.track_programme(P(integrator, 0.5), z0, d0, np.full(500, a), np.zeros(500))
    zb, db = oracle.track(P(integrator, 0.5, voltage_V=a * wl.RING["voltage_V"]), z0, d0, 500)
    assert np.max(np.abs(za - zb)) <= 1e-12 and np.max(np.abs(da - db)) <= 1e-14


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_constant_phase_offset_is_a_shift_of_the_origin(integrator):
    """sin(kappa z + psi) = sin(kappa (z + psi/kappa)): tracking with a constant offset is
    tracking the shifted coordinate z + psi/kappa without one (both harmonics, G28)."""
    p = P(integrator, 0.5)
    kappa = oracle.derive(p)["kappa"]
    z0, d0 = small_bunch()
    psi = 0.4
    za, da = oracle.track_programme(p, z0, d0, np.ones(400), np.full(400, psi))
    zb, db = oracle.track(p, z0 + psi / kappa, d0, 400)
    assert np.max(np.abs(za + psi / kappa - zb)) <= 1e-11
    assert np.max(np.abs(da - db)) <= 1e-13


def test_impulse_programme_kicks_exactly_once_at_the_right_turn():
    """a_t = 0 except at t = 6: delta stays put for turns 1..6, changes at turn 7 only."""
    p = P("leapfrog")
    a = np.zeros(10)
    a[6] = 1.0
    z0, d0 = np.array([0.2]), np.array([1e-3])
    for t in range(1, 11):
        _, d = oracle.track_programme(p, z0, d0, a[:t], np.zeros(t))
        assert (d[0] == d0[0]) == (t <= 6), t
    # and the one kick is F(z) at the drifted position
    g = oracle.derive(p)
    z_at_kick = 0.2 - 13 * g["d"] * 1e-3            # 6 full turns of drift + the leading half
    _, d = oracle.track_programme(p, z0, d0, a[:7], np.zeros(7))
    assert d[0] - d0[0] == pytest.approx(g["A"] * math.sin(g["kappa"] * z_at_kick), rel=1e-12)


def test_slow_voltage_ramp_conserves_the_emittance():
    """Adiabatic invariance: for small amplitudes sigma_z ~ V^(-1/4), sigma_delta ~ V^(1/4)
    when V changes slowly compared with the synchrotron period (169 turns)."""
    p = P("leapfrog")
    z0, d0 = wl.gaussian_bunch(4000, 0.02, 11)
    turns, ratio = 20000, 4.0
    a = np.linspace(1.0, ratio, turns)
    z, d = oracle.track_programme(p, z0, d0, a, np.zeros(turns))
    m0, m1 = oracle.moments_of(p, z0, d0), oracle.moments_of(p, z, d)
    assert m1["rms_z"] / m0["rms_z"] == pytest.approx(ratio ** -0.25, rel=1e-2)
    assert m1["rms_d"] / m0["rms_d"] == pytest.approx(ratio ** 0.25, rel=1e-2)
    assert m1["rms_z"] * m1["rms_d"] == pytest.approx(m0["rms_z"] * m0["rms_d"], rel=5e-3)


def test_resonant_phase_modulation_drives_the_dipole_mode():
    """psi_t = eps sin(mu t) at the synchrotron tune pumps the centroid linearly in time:
    after N turns |<z>| ~ eps N / (2 kappa) (driven harmonic oscillator at resonance), while
    the same modulation far off resonance leaves it at the eps/kappa level."""
    p = P("leapfrog")
    g = oracle.derive(p)
    mu = math.acos(1 - g["K"] / 2)
    z0, d0 = wl.gaussian_bunch(2000, 0.01, 5)
    eps, N = 1e-3, 845                      # 5 synchrotron periods
    t = np.arange(N)
    amp = []
    for tune in (mu, 3.3 * mu):
        _, _, mom = oracle.track_programme_moments(p, z0, d0, np.ones(N), eps * np.sin(tune * t))
        amp.append(np.max(np.abs(mom["mean_z"][-170:])))
    # z'' + mu^2 z = -(mu^2 / kappa) psi(n)  =>  resonant amplitude eps mu n / (2 kappa)
    assert amp[0] == pytest.approx(eps * mu * N / (2 * g["kappa"]), rel=0.1)
    assert amp[1] < 5 * eps / g["kappa"]


def test_programme_fp64_against_80_bit_twin():
    p = P("ruth4", 0.5)
    z0, d0 = small_bunch(64, sigma_z=0.1)
    rng = np.random.default_rng(2)
    # gentle noise: a violent programme heats particles out of the bucket, where rounding
    # differences are amplified (G17) and the comparison says nothing about the arithmetic
    a, psi = rng.uniform(0.9, 1.1, 1000), rng.uniform(-0.05, 0.05, 1000)
    z, d = oracle.track_programme(p, z0, d0, a, psi)
    zl, dl = oracle.track_programme_ld(p, z0, d0, a, psi)
    assert np.max(np.abs(z)) < 0.7
    g = oracle.derive(p)
    assert np.max(np.abs(z - zl.astype(np.float64))) / g["z_max"] < 1e-11
    assert np.max(np.abs(d - dl.astype(np.float64))) / 2.6e-3 < 1e-11


def test_programme_moments_index():
    p = P("leapfrog")
    z0, d0 = small_bunch(500)
    rng = np.random.default_rng(8)
    a, psi = rng.uniform(0.5, 1.5, 12), rng.uniform(-0.5, 0.5, 12)
    _, _, mom = oracle.track_programme_moments(p, z0, d0, a, psi)
    for t in (1, 5, 12):
        z, d = oracle.track_programme(p, z0, d0, a[:t], psi[:t])
        assert mom["mean_z"][t - 1] == oracle.moments_of(p, z, d)["mean_z"]


# ================================================================== f4: slicing
def test_slices_exact_edges_on_a_dyadic_grid():
    """[-1, 1) in 8 slices: edges are multiples of 1/4, every operation is exact.  Left-closed,
    right-open slices; z_hi itself, +inf and NaN are 'above'; -inf and < z_lo are 'below'."""
    z = np.array([-1.0, -0.75, -0.7500000000000001, 0.0, 0.25, 0.24999999999999997, 0.999999,
                  1.0, 1.5, -1.0000000000000002, np.inf, -np.inf, np.nan, -0.0])
    h = oracle.slice_histogram(z, -1.0, 1.0, 8)
    expect = np.zeros(10, dtype=np.uint64)
    expect[0] = 2                      # -1.0000000000000002, -inf
    expect[9] = 4                      # 1.0, 1.5, +inf, nan
    expect[1 + 0] = 2                  # -1.0, -0.7500000000000001
    expect[1 + 1] = 1                  # -0.75
    expect[1 + 4] = 2                  # 0.0, -0.0
    # 0.24999999999999997 + 1 rounds to 1.25, so the RULE (decision taken in fp64 on
    # (z - z_lo) * inv, G29) puts it into slice 5 together with 0.25
    expect[1 + 5] = 2
    expect[1 + 7] = 1                  # 0.999999
    assert np.array_equal(h, expect), (h, expect)
    assert h.sum() == z.size


def test_slices_match_numpy_histogram_on_seeded_data():
    rng = np.random.default_rng(12)
    z = rng.normal(0.0, 0.23, 200_000)
    zmax = oracle.derive(P())["z_max"]
    for S in (1, 7, 64, 1000):
        h = oracle.slice_histogram(z, -zmax, zmax, S)
        ref, _ = np.histogram(z[(z >= -zmax) & (z < zmax)], bins=S, range=(-zmax, zmax))
        assert np.array_equal(h[1:-1], ref.astype(np.uint64)), S
        assert h[0] == np.sum(z < -zmax) and h[-1] == np.sum(z >= zmax)


def test_slices_brute_force_and_the_upper_clamp():
    """Pure-Python restatement on a tiny input; and a range whose upper edge rounds u up to S."""
    rng = np.random.default_rng(4)
    z = rng.uniform(-0.3, 1.3, 500)
    lo, hi, S = 0.1, 1.0, 9
    h = oracle.slice_histogram(z, lo, hi, S)
    ref = [0] * (S + 2)
    inv = S / (hi - lo)
    for v in z:
        if v < lo:
            ref[0] += 1
        elif not v < hi:
            ref[S + 1] += 1
        else:
            ref[1 + min(int(math.floor((v - lo) * inv)), S - 1)] += 1
    assert list(h) == ref
    # largest double below z_hi with S = 3 over [0, 0.3): (z - 0) * (3/0.3) rounds to 3.0 -> clamp
    zhi = 0.3
    zl = np.nextafter(zhi, 0.0)
    assert math.floor((zl - 0.0) * (3 / (zhi - 0.0))) in (2, 3)
    h = oracle.slice_histogram(np.array([zl]), 0.0, zhi, 3)
    assert list(h) == [0, 0, 0, 1, 0]


def test_track_slices_index_and_conservation():
    p = P("leapfrog")
    z0, d0 = small_bunch(3000)
    zmax = oracle.derive(p)["z_max"]
    z, d, h = oracle.track_slices(p, z0, d0, 7, -zmax, zmax, 32)
    assert h.shape == (7, 34) and np.all(h.sum(axis=1) == 3000)
    for t in (1, 4, 7):
        zt, _ = oracle.track(p, z0, d0, t)
        assert np.array_equal(h[t - 1], oracle.slice_histogram(zt, -zmax, zmax, 32))
    zt, dt = oracle.track(p, z0, d0, 7)
    assert np.array_equal(z, zt) and np.array_equal(d, dt)


# ================================================================== f3: transverse maps
def twiss_matrix(alpha, beta, mu):
    """Textbook periodic Courant-Snyder matrix (typed here, not taken from the product)."""
    gam = (1 + alpha * alpha) / beta
    c, s = math.cos(mu), math.sin(mu)
    return np.array([[c + alpha * s, beta * s], [-gam * s, c - alpha * s]])


def block4(mx, my):
    m = np.zeros((4, 4))
    m[:2, :2] = mx
    m[2:, 2:] = my
    return m


def coords(n=300, seed=1):
    rng = np.random.default_rng(seed)
    return (rng.normal(0, 1e-3, n), rng.normal(0, 2e-5, n), rng.normal(0, 8e-4, n),
            rng.normal(0, 1.5e-5, n))


def test_transverse_small_integer_matrix_exact():
    """M = [[1,1,0,0],[0,1,0,0],[0,0,1,2],[3,0,0,1]] is not symmetric: a transposed or
    column-major reading fails.  All arithmetic is exact on small integers."""
    M = np.array([[1, 1, 0, 0], [0, 1, 0, 0], [0, 0, 1, 2], [3, 0, 0, 1]], dtype=float)
    x, xp, y, yp = np.array([1.0]), np.array([2.0]), np.array([3.0]), np.array([4.0])
    out = oracle.track_transverse(P(), [M], x, xp, y, yp, None, None, 1)
    assert [float(a[0]) for a in out[:4]] == [3.0, 2.0, 11.0, 7.0]
    out = oracle.track_transverse(P(), [M], x, xp, y, yp, None, None, 3)
    ref = np.linalg.matrix_power(M, 3) @ np.array([1.0, 2.0, 3.0, 4.0])
    assert [float(a[0]) for a in out[:4]] == list(ref)


def test_transverse_periodic_twiss_matrix_power_closed_form():
    """N turns through the one-turn Courant-Snyder matrix equal ONE application of the same
    matrix with phase advance N mu (de Moivre for the Twiss matrix), and the Courant-Snyder
    invariant gamma x^2 + 2 alpha x x' + beta x'^2 is conserved."""
    ax, bx, mux = -0.8, 54.6, 2 * math.pi * 0.13
    ay, by, muy = 0.5, 48.2, 2 * math.pi * 0.18
    M = block4(twiss_matrix(ax, bx, mux), twiss_matrix(ay, by, muy))
    x, xp, y, yp = coords()
    N = 1000
    out = oracle.track_transverse(P(), [M], x, xp, y, yp, None, None, N)
    MN = block4(twiss_matrix(ax, bx, N * mux), twiss_matrix(ay, by, N * muy))
    ref = MN @ np.vstack([x, xp, y, yp])
    for k, scale in enumerate((1e-3, 2e-5, 8e-4, 1.5e-5)):
        assert np.max(np.abs(out[k] - ref[k])) <= 1e-11 * scale, k
    gx = (1 + ax * ax) / bx
    J0 = gx * x * x + 2 * ax * x * xp + bx * xp * xp
    J1 = gx * out[0] ** 2 + 2 * ax * out[0] * out[1] + bx * out[1] ** 2
    assert np.max(np.abs(J1 / J0 - 1)) <= 1e-11


def test_transverse_segment_order_and_coupling():
    """Two non-commuting segments (a rotation and a thin skew quadrupole that couples x and y):
    one turn is M_1 M_0, not M_0 M_1; N turns equal numpy's matrix power."""
    M0 = block4(twiss_matrix(0.3, 20.0, 1.1), twiss_matrix(-0.2, 35.0, 0.7))
    M1 = np.eye(4)
    M1[1, 2] = 1e-2            # x' += k y
    M1[3, 0] = 1e-2            # y' += k x
    assert not np.allclose(M1 @ M0, M0 @ M1)
    x, xp, y, yp = coords(50)
    u = np.vstack([x, xp, y, yp])
    out = oracle.track_transverse(P(), [M0, M1], x, xp, y, yp, None, None, 1)
    assert np.allclose(np.vstack(out[:4]), M1 @ M0 @ u, rtol=1e-13, atol=1e-20)
    assert not np.allclose(np.vstack(out[:4]), M0 @ M1 @ u, rtol=1e-6, atol=1e-12)
    out = oracle.track_transverse(P(), [M0, M1], x, xp, y, yp, None, None, 200)
    ref = np.linalg.matrix_power(M1 @ M0, 200) @ u
    assert np.allclose(np.vstack(out[:4]), ref, rtol=1e-10, atol=1e-16)


def test_transverse_identity_and_decoupled_longitudinal_plane():
    p = P("leapfrog")
    x, xp, y, yp = coords(100)
    z0, d0 = small_bunch(100)
    out = oracle.track_transverse(p, [np.eye(4)] * 3, x, xp, y, yp, z0, d0, 50)
    assert all(np.array_equal(a, b) for a, b in zip(out[:4], (x, xp, y, yp)))
    zt, dt = oracle.track(p, z0, d0, 50)
    assert np.array_equal(out[4], zt) and np.array_equal(out[5], dt)
