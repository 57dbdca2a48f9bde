"""Pins of the CPU oracle against what the paper's physics and the mathematics fix
(BASELINE.json:north_star (3); SURVEY.md sec. 8(c) "What pins the oracle").

None of these tests touches the CUDA path.  Each is chosen so that a plausible mistake in
oracle/ (dropped term, wrong sign, wrong coefficient, transposed operand, wrong sub-step
order) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
from scipy.special import ellipk

import oracle
from paper_1610_05801_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
INTEGRATORS = ("euler_cromer", "leapfrog", "ruth4")
# exact cubic of the Forest-Ruth linearised half-trace
RUTH_K3 = 0.064754199504677651815


def P(integrator="leapfrog", ratio2=0.0, **ring_over):
    ring = dict(wl.RING)
    ring.update(ring_over)
    return oracle.make_params(ring, integrator, ratio2)


def golden_constants():
    out = {}
    for line in open(os.path.join(GOLD, "derived_constants.txt")):
        if line.startswith("#"):
            continue
        k, v = line.split()
        out[k] = float(v)
    return out


def half_trace_closed_form(integrator, K):
    if integrator == "ruth4":
        return 1.0 - K / 2 + K * K / 24 + RUTH_K3 * K ** 3
    return 1.0 - K / 2


# ---------------------------------------------------------------- derived constants
def test_derived_constants_match_40_digit_values():
    g = golden_constants()
    d = oracle.derive(P())
    for k in ("R", "beta", "eta", "A", "d", "kappa", "K", "z_max", "H_sep"):
        assert abs(d[k] - g[k]) <= 4 * np.spacing(abs(g[k])), k
    # BASELINE.json:configs[0] quotes eta ~ 6.2e-4, A ~ 7.7e-5, Q_s ~ 0.006
    assert round(d["eta"], 5) == 6.2e-4 and round(d["A"], 6) == 7.7e-5
    assert abs(math.acos(1 - d["K"] / 2) / (2 * math.pi) - 0.006) < 1e-4


# ---------------------------------------------------------------- hand-iterated values
def test_hand_iterated_values():
    """40-digit hand iteration of the stated map (tests/golden/hand_values.txt)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "hand_values.txt")) if l[0] != "#"]
    assert len(rows) == 3 * 2 * 4 * 3
    for name, r, z0, d0, t, z_ref, d_ref in rows:
        z, d = oracle.track(P(name, float(r)), [float(z0)], [float(d0)], int(t))
        z_ref, d_ref = float(z_ref), float(d_ref)
        # <= 1e-14 relative after 3 turns, <= 1e-11 after 1000
        tol = 1e-14 if int(t) <= 3 else 1e-11
        assert abs(z[0] - z_ref) <= tol * max(abs(z_ref), 0.1), (name, r, z0, d0, t)
        assert abs(d[0] - d_ref) <= tol * max(abs(d_ref), 1e-3), (name, r, z0, d0, t)


def test_hand_iterated_values_with_synchronous_phase():
    """Reading G3, F(z) = A[sin(phi_s + kappa z) - sin(phi_s) + r sin(2 kappa z)], iterated by
    hand in 40 digits at phi_s = 0.3 and -0.7 (tests/golden/phi_s_values.txt, mpmath only).
    The linear half-trace pin below sees only cos(phi_s): this one fails on a flipped sign of
    phi_s, a missing - sin(phi_s), phi_s leaking into the 2h term, or any stand-in that merely
    agrees to first order (e.g. cos(phi_s) sin(kappa z))."""
    rows = [l.split() for l in open(os.path.join(GOLD, "phi_s_values.txt")) if l[0] != "#"]
    assert len(rows) == 3 * 2 * 2 * 4 * 3
    seen = set()
    for name, phi, r, z0, d0, t, z_ref, d_ref in rows:
        p = oracle.make_params(wl.RING, name, float(r), phi_s=float(phi))
        z, d = oracle.track(p, [float(z0)], [float(d0)], int(t))
        z_ref, d_ref = float(z_ref), float(d_ref)
        tol = 1e-14 if int(t) <= 3 else 1e-11
        assert abs(z[0] - z_ref) <= tol * max(abs(z_ref), 0.1), (name, phi, r, z0, d0, t)
        assert abs(d[0] - d_ref) <= tol * max(abs(d_ref), 1e-3), (name, phi, r, z0, d0, t)
        seen.add((name, phi, r))
    assert len(seen) == 12


def test_synchronous_phase_values_discriminate_the_plausible_mistakes():
    """The golden values above are far (>= 1e-8) from what the wrong formulas give after one
    turn, so the 1e-14 gate separates them: sign of phi_s, dropped sin(phi_s), first-order
    stand-in.  Evaluated here in plain Python floats from the golden constants."""
    g = golden_constants()
    rows = [l.split() for l in open(os.path.join(GOLD, "phi_s_values.txt")) if l[0] != "#"]
    for name, phi, r, z0, d0, t, z_ref, d_ref in rows:
        if name != "euler_cromer" or t != "1":
            continue
        phi, r, z0, d0, d_ref = float(phi), float(r), float(z0), float(d0), float(d_ref)
        kz = g["kappa"] * z0
        right = d0 + g["A"] * (math.sin(phi + kz) - math.sin(phi) + r * math.sin(2 * kz))
        assert abs(right - d_ref) <= 1e-15
        wrong = (d0 + g["A"] * (math.sin(-phi + kz) - math.sin(-phi) + r * math.sin(2 * kz)),
                 d0 + g["A"] * (math.sin(phi + kz) + r * math.sin(2 * kz)),
                 d0 + g["A"] * (math.cos(phi) * math.sin(kz) + r * math.sin(2 * kz)),
                 d0 + g["A"] * (math.sin(phi + kz) - math.sin(phi) + r * math.sin(2 * (kz + phi))))
        if r == 0.0:
            wrong = wrong[:3]             # no 2h term for phi_s to leak into
        if z0 != 0.0:
            assert all(abs(w - d_ref) >= 1e-8 for w in wrong), (phi, r, z0)


def test_first_hand_value_by_pocket_calculator():
    """(z, delta) = (0.1, 0): the first half drift leaves z, the kick is A sin(kappa*0.1),
    the second half drift subtracts d times it."""
    g = golden_constants()
    z, d = oracle.one_turn(P(), [0.1], [0.0])
    kick = g["A"] * math.sin(g["kappa"] * 0.1)
    assert d[0] == pytest.approx(kick, rel=1e-15)
    assert z[0] == pytest.approx(0.1 - g["d"] * kick, rel=1e-15)


# ---------------------------------------------------------------- linear tune, det
@pytest.mark.parametrize("integrator", INTEGRATORS)
@pytest.mark.parametrize("ratio2", [0.0, 0.5, -0.25])
def test_linearised_map_has_exact_discrete_tune(integrator, ratio2):
    """cos(mu) = 1 - K/2 with K = eta*C*A*h/R (north_star (3)); K -> K(1+2r) for the
    double harmonic; the Ruth4 half-trace is an exact cubic in K (G9)."""
    p = P(integrator, ratio2)
    K = golden_constants()["K"] * (1 + 2 * ratio2)
    ez, ed = 1e-7, 1e-9
    za, da = oracle.one_turn(p, [ez], [0.0])
    zb, db = oracle.one_turn(p, [0.0], [ed])
    M = np.array([[za[0] / ez, zb[0] / ed], [da[0] / ez, db[0] / ed]])
    assert abs(0.5 * np.trace(M) - half_trace_closed_form(integrator, K)) <= 1e-12
    assert abs(np.linalg.det(M) - 1.0) <= 1e-12


def test_leapfrog_matrix_entries():
    """M = [[1-dk, -d(2-dk)], [k, 1-dk]], k = A*kappa (product of the three shears)."""
    g = golden_constants()
    d, k = g["d"], g["A"] * g["kappa"]
    ez, ed = 1e-7, 1e-9
    za, da = oracle.one_turn(P(), [ez], [0.0])
    zb, db = oracle.one_turn(P(), [0.0], [ed])
    M = np.array([[za[0] / ez, zb[0] / ed], [da[0] / ez, db[0] / ed]])
    ref = np.array([[1 - d * k, -d * (2 - d * k)], [k, 1 - d * k]])
    assert np.allclose(M, ref, rtol=1e-10, atol=0)


def test_phi_s_scales_linear_focusing_by_cos():
    """Reading G3: F(z) = A[sin(phi_s+kappa z) - sin phi_s]  =>  K -> K cos(phi_s)."""
    g = golden_constants()
    for phi_s in (0.3, -0.7):
        p = oracle.make_params(wl.RING, "leapfrog", 0.0, phi_s=phi_s)
        ez, ed = 1e-8, 1e-10
        za, da = oracle.one_turn(p, [ez], [0.0])
        zb, db = oracle.one_turn(p, [0.0], [ed])
        half_tr = 0.5 * (za[0] / ez + db[0] / ed)
        assert abs(half_tr - (1 - g["K"] * math.cos(phi_s) / 2)) <= 1e-10
        assert oracle.kick(p, 0.0) == 0.0


def test_order_of_accuracy_of_the_tune():
    """|mu - sqrt(K)| ~ K^(3/2)/24 for the 2nd-order maps, ~K^(5/2) level for Ruth4."""
    K = golden_constants()["K"]
    mu2 = math.acos(half_trace_closed_form("leapfrog", K))
    mu4 = math.acos(half_trace_closed_form("ruth4", K))
    assert abs(mu2 - math.sqrt(K)) == pytest.approx(K ** 1.5 / 24, rel=1e-3)
    assert abs(mu4 - math.sqrt(K)) < 1e-8 < abs(mu2 - math.sqrt(K)) / 100


# ---------------------------------------------------------------- symplecticity
@pytest.mark.parametrize("integrator", INTEGRATORS)
@pytest.mark.parametrize("ratio2", [0.0, 0.5])
def test_one_turn_jacobian_determinant_is_one(integrator, ratio2):
    """Finite-difference Jacobian of the oracle's one-turn map at 100 random in-bucket
    points: |det - 1| <= 1e-7 (central differences)."""
    p = P(integrator, ratio2)
    rng = np.random.default_rng(7)
    z0 = rng.uniform(-0.7, 0.7, 100)
    d0 = rng.uniform(-3e-3, 3e-3, 100)
    hz, hd = 1e-6, 1e-8
    zp, dp = oracle.one_turn(p, z0 + hz, d0)
    zm, dm = oracle.one_turn(p, z0 - hz, d0)
    zq, dq = oracle.one_turn(p, z0, d0 + hd)
    zr, dr = oracle.one_turn(p, z0, d0 - hd)
    det = ((zp - zm) / (2 * hz)) * ((dq - dr) / (2 * hd)) \
        - ((zq - zr) / (2 * hd)) * ((dp - dm) / (2 * hz))
    assert np.max(np.abs(det - 1.0)) <= 1e-7


def test_leapfrog_jacobian_matches_product_of_shears():
    """Analytic Jacobian = D * Kick'(z_mid) * D (each a shear of determinant 1)."""
    g = golden_constants()
    p = P("leapfrog", 0.5)
    rng = np.random.default_rng(8)
    z0 = rng.uniform(-0.7, 0.7, 20)
    d0 = rng.uniform(-3e-3, 3e-3, 20)
    hz, hd = 1e-6, 1e-8
    zp, dp = oracle.one_turn(p, z0 + hz, d0)
    zm, dm = oracle.one_turn(p, z0 - hz, d0)
    zq, dq = oracle.one_turn(p, z0, d0 + hd)
    zr, dr = oracle.one_turn(p, z0, d0 - hd)
    for i in range(z0.size):
        zmid = z0[i] - g["d"] * d0[i]
        fp = g["A"] * g["kappa"] * (math.cos(g["kappa"] * zmid)
                                    + 2 * 0.5 * math.cos(2 * g["kappa"] * zmid))
        D = np.array([[1.0, -g["d"]], [0.0, 1.0]])
        Km = np.array([[1.0, 0.0], [fp, 1.0]])
        J = D @ Km @ D
        Jfd = np.array([[(zp[i] - zm[i]) / (2 * hz), (zq[i] - zr[i]) / (2 * hd)],
                        [(dp[i] - dm[i]) / (2 * hz), (dq[i] - dr[i]) / (2 * hd)]])
        assert np.allclose(J, Jfd, rtol=2e-6, atol=1e-9)
        assert abs(np.linalg.det(J) - 1) < 1e-14


# ---------------------------------------------------------------- time reversal
@pytest.mark.parametrize("integrator", ["leapfrog", "ruth4"])
@pytest.mark.parametrize("ratio2", [0.0, 0.5])
def test_time_reversal(integrator, ratio2):
    """Forward N turns, delta -> -delta, forward N turns, delta -> -delta returns to the
    start within rounding (LF and Ruth4 are self-adjoint, G24)."""
    p = P(integrator, ratio2)
    z_max = golden_constants()["z_max"]
    rng = np.random.default_rng(0)
    z0 = rng.uniform(-0.6, 0.6, 1000)
    d0 = rng.uniform(-2e-3, 2e-3, 1000)
    inb = oracle.bucket_mask(p, z0, d0)
    z, d = oracle.track(p, z0, d0, 1000)
    z, d = oracle.track(p, z, -d, 1000)
    d = -d
    assert inb.sum() > 500
    assert np.max(np.abs(z - z0)[inb]) <= 1e-10 * z_max
    assert np.max(np.abs(d - d0)[inb]) <= 1e-10 * 2e-3


def test_euler_cromer_reverses_only_through_its_adjoint():
    """EC (kick, drift) is not self-adjoint: its time reverse is (drift, kick) (G24)."""
    p = P("euler_cromer")
    z_max = golden_constants()["z_max"]
    rng = np.random.default_rng(1)
    z0 = rng.uniform(-0.5, 0.5, 200)
    d0 = rng.uniform(-1.5e-3, 1.5e-3, 200)
    z, d = oracle.track(p, z0, d0, 500)
    d = -d
    for _ in range(500):
        z, d = oracle.one_turn_ec_adjoint(p, z, d)
    assert np.max(np.abs(z - z0)) <= 1e-10 * z_max
    assert np.max(np.abs(-d - d0)) <= 1e-10 * 2e-3
    # the naive self-reverse does NOT come back
    z, d = oracle.track(p, z0, d0, 500)
    z, d = oracle.track(p, z, -d, 500)
    assert np.max(np.abs(z - z0)) > 1e-4 * z_max


# ---------------------------------------------------------------- Hamiltonian
def h_oscillation(p, z0, turns, every=1):
    z = np.array(z0, dtype=float)
    d = np.zeros_like(z)
    H0 = oracle.hamiltonian(p, z, d)
    worst = np.zeros_like(z)
    done = 0
    while done < turns:
        z, d = oracle.track(p, z, d, every)
        done += every
        worst = np.maximum(worst, np.abs(oracle.hamiltonian(p, z, d) / H0 - 1))
    return worst


def test_hamiltonian_bounded_no_secular_drift():
    """max|H/H0 - 1| over 10^4 turns equals that over 4*10^4 turns (no secular drift),
    and its size orders the integrators: EC ~ sqrt(K)/2 >> LF ~ K/4 >> Ruth4."""
    z0 = [0.01, 0.1, 0.3, 0.5, 0.65, 0.72]
    K = golden_constants()["K"]
    amp = {}
    for name in INTEGRATORS:
        p = P(name)
        a = h_oscillation(p, z0, 10_000)
        b = h_oscillation(p, z0, 40_000, every=1 if name != "ruth4" else 1)
        assert np.all(b >= a * (1 - 1e-12))
        # the oscillation amplitude is already saturated after 10^4 turns (59 periods)
        assert np.allclose(a, b, rtol=2e-2 if name == "ruth4" else 5e-3), (name, a, b)
        amp[name] = a
    assert amp["leapfrog"][0] == pytest.approx(K / 4, rel=2e-2)       # 3.45e-4
    assert amp["euler_cromer"][0] == pytest.approx(math.sqrt(K) / 2, rel=3e-2)  # 1.9e-2
    assert np.all(amp["ruth4"] < 2e-7)
    assert np.all(amp["euler_cromer"] > 30 * amp["leapfrog"])
    assert np.all(amp["leapfrog"] > 500 * amp["ruth4"])
    # SURVEY.md 8(c) item 4 probe values for LF
    assert np.allclose(amp["leapfrog"], [3.45e-4, 3.35e-4, 2.65e-4, 1.72e-4, 1.24e-4, 1.16e-4],
                       rtol=2e-2)


def test_double_harmonic_hamiltonian_is_conserved_too():
    """Ties the r-term of H to the r-term of the kick: with r = 0.5 a wrong factor in
    either makes H oscillate at the 10^-1 level instead of 10^-3."""
    p = P("leapfrog", 0.5)
    a = h_oscillation(p, [0.05, 0.2, 0.4, 0.6], 3000)
    assert np.all(a < 1.5e-3)
    p4 = P("ruth4", 0.5)
    assert np.all(h_oscillation(p4, [0.05, 0.2, 0.4, 0.6], 3000) < 2e-6)


def test_hamiltonian_special_points():
    g = golden_constants()
    p = P()
    assert oracle.hamiltonian(p, 0.0, 0.0)[0] == 0.0
    # unstable fixed point (+-z_max, 0) and top of the separatrix (0, delta_max) sit on H_sep
    assert oracle.hamiltonian(p, g["z_max"], 0.0)[0] == pytest.approx(g["H_sep"], rel=1e-14)
    assert oracle.hamiltonian(p, 0.0, g["delta_max"])[0] == pytest.approx(g["H_sep"], rel=1e-14)
    # the r-term vanishes at kappa z = pi: same H_sep with the second harmonic
    assert oracle.hamiltonian(P(ratio2=0.5), g["z_max"], 0.0)[0] == pytest.approx(
        g["H_sep"], rel=1e-14)
    # small-amplitude: H -> eta C delta^2/2 + A kappa (1+2r) z^2 / 2
    z, r = 1e-4, 0.5
    assert oracle.hamiltonian(P(ratio2=r), z, 0.0)[0] == pytest.approx(
        0.5 * g["A"] * g["kappa"] * (1 + 2 * r) * z * z, rel=1e-6)


# ---------------------------------------------------------------- pendulum period
@pytest.mark.parametrize("integrator,tol", [("leapfrog", 2e-4), ("euler_cromer", 2e-4),
                                             ("ruth4", 2e-6)])
def test_nonlinear_period_matches_elliptic_integral(integrator, tol):
    """The continuous limit is a pendulum: T(z_hat) = (2 pi / sqrt(K)) * (2/pi) K_ell(m),
    m = sin^2(kappa z_hat / 2).  Measured from the oracle's zero crossings over many
    periods.  A wrong kappa, A, d or sin argument shifts it at the 10^-1 level; the
    discrete maps differ from the pendulum by O(K) (2nd order) / O(K^2) (Ruth4)."""
    g = golden_constants()
    p = P(integrator)
    for z_hat in (0.05, 0.4, 0.65):
        m = math.sin(g["kappa"] * z_hat / 2) ** 2
        T_ref = (2 * math.pi / math.sqrt(g["K"])) * (2 / math.pi) * ellipk(m)
        z, d = np.array([z_hat]), np.array([0.0])
        turns = int(40 * T_ref)
        zs = np.empty(turns + 1)
        zs[0] = z_hat
        for t in range(turns):
            z, d = oracle.one_turn(p, z, d)
            zs[t + 1] = z[0]
        # downward zero crossings, linearly interpolated
        idx = np.where((zs[:-1] > 0) & (zs[1:] <= 0))[0]
        tc = idx + zs[idx] / (zs[idx] - zs[idx + 1])
        T = (tc[-1] - tc[0]) / (len(tc) - 1)
        assert abs(T / T_ref - 1) < tol, (integrator, z_hat, T, T_ref)


# ---------------------------------------------------------------- special cases
def test_no_rf_is_a_pure_shear():
    """A = 0 (V = 0): z -> z - eta*C*delta*N exactly up to rounding, delta untouched."""
    g = golden_constants()
    for name in INTEGRATORS:
        p = P(name, voltage_V=0.0)
        z0 = np.array([0.3, -0.2, 0.0])
        d0 = np.array([1e-3, -2e-3, 5e-4])
        z, d = oracle.track(p, z0, d0, 1000)
        assert np.array_equal(d, d0)
        assert np.allclose(z, z0 - 2 * g["d"] * 1000 * d0, rtol=1e-12, atol=0)


def test_no_slippage_is_a_fixed_kick_per_turn():
    """eta = 0 (alpha_c = 1/gamma^2): z never moves, delta grows by F(z) per turn."""
    ring = dict(wl.RING)
    ring["alpha_c"] = 1.0 / ring["gamma"] ** 2
    for name in INTEGRATORS:
        p = oracle.make_params(ring, name, 0.5)
        assert oracle.derive(p)["eta"] == 0.0
        z0 = np.array([0.3, -0.2])
        z, d = oracle.track(p, z0, [0.0, 0.0], 100)
        assert np.array_equal(z, z0)
        F = np.array([oracle.kick(p, zz) for zz in z0])
        assert np.allclose(d, 100 * F, rtol=1e-12)


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_small_amplitude_is_the_linear_map_to_the_nth_power(integrator):
    """At amplitude 1e-7 m the map is its own linearisation: N turns = M^N (numpy)."""
    p = P(integrator)
    ez, ed = 1e-7, 1e-9
    za, da = oracle.one_turn(p, [ez], [0.0])
    zb, db = oracle.one_turn(p, [0.0], [ed])
    M = np.array([[za[0] / ez, zb[0] / ed], [da[0] / ez, db[0] / ed]])
    v0 = np.array([0.6e-7, -0.8e-9 * 0.3])
    z, d = oracle.track(p, [v0[0]], [v0[1]], 500)
    ref = np.linalg.matrix_power(M, 500) @ v0
    assert z[0] == pytest.approx(ref[0], rel=1e-6, abs=1e-15)
    assert d[0] == pytest.approx(ref[1], rel=1e-6, abs=1e-18)
    # and the rotation angle per turn is mu
    K = golden_constants()["K"]
    mu = math.acos(half_trace_closed_form(integrator, K))
    lam = np.linalg.eigvals(M)
    assert abs(abs(np.angle(lam[0])) - mu) < 1e-9


def test_kick_function():
    g = golden_constants()
    p = P(ratio2=0.5)
    for z in (0.05, -0.3, 0.7, 12.3, -1500.0):
        ph = g["kappa"] * z
        ref = g["A"] * (math.sin(ph) + 0.5 * math.sin(2 * ph))
        # the phase kappa*z carries a rounding of |ph|*2^-53 (matters at |z| = 1500 m)
        assert abs(oracle.kick(p, z) - ref) <= g["A"] * (4e-16 * abs(ph) + 1e-15)
    # odd, and zero at the fixed points
    assert oracle.kick(p, 0.3) == -oracle.kick(p, -0.3)
    assert abs(oracle.kick(P(), g["z_max"])) < 1e-19


# ---------------------------------------------------------------- 80-bit self-check
@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_fp64_oracle_against_its_80_bit_twin(integrator):
    """Bounds the fp64 oracle's own rounding after 1000 turns:
    <= 1e-11 of z_max / sigma_delta away from the separatrix layer."""
    cfg = wl.CONFIGS[0]
    z0, d0 = wl.make_bunch(cfg)
    p = P(integrator)
    g = golden_constants()
    z, d = oracle.track(p, z0, d0, 1000)
    zl, dl = oracle.track_ld(p, z0, d0, 1000)
    H0 = oracle.hamiltonian(p, z0, d0)
    away = np.abs(1 - H0 / g["H_sep"]) > 1e-2
    sd = wl.matched_sigma_delta(cfg["sigma_z"])
    ez = np.abs((z.astype(np.longdouble) - zl).astype(float)) / g["z_max"]
    ed = np.abs((d.astype(np.longdouble) - dl).astype(float)) / sd
    assert away.sum() > 900
    assert ez[away].max() < 1e-11 and ed[away].max() < 1e-11


# ---------------------------------------------------------------- moments, membership
def test_moments_against_numpy():
    rng = np.random.default_rng(3)
    z = rng.normal(0.01, 0.2, 10_000)
    d = rng.normal(-1e-5, 2e-3, 10_000)
    m = oracle.moments_of(P(), z, d)
    zl, dl = z.astype(np.longdouble), d.astype(np.longdouble)
    assert m["mean_z"] == pytest.approx(float(zl.mean()), rel=1e-14)
    assert m["mean_d"] == pytest.approx(float(dl.mean()), rel=1e-14)
    assert m["rms_z"] == pytest.approx(float(zl.std()), rel=1e-14)     # population (ddof=0)
    assert m["rms_d"] == pytest.approx(float(dl.std()), rel=1e-14)
    assert m["cov_zd"] == pytest.approx(float(((zl - zl.mean()) * (dl - dl.mean())).mean()),
                                        rel=1e-12)
    # a shifted bunch: rms is about the mean, not about zero
    m2 = oracle.moments_of(P(), z + 5.0, d)
    assert m2["rms_z"] == pytest.approx(m["rms_z"], rel=1e-12)
    assert m2["mean_z"] == pytest.approx(m["mean_z"] + 5.0, rel=1e-14)


def test_track_moments_indexing():
    """moments[t] is the state after turn t+1 and the final arrays are the N-turn state."""
    p = P()
    z0, d0 = wl.make_bunch(wl.CONFIGS[0], n=200)
    z, d, mom = oracle.track_moments(p, z0, d0, 5)
    for t in range(5):
        zt, dt = oracle.track(p, z0, d0, t + 1)
        assert mom["mean_z"][t] == pytest.approx(zt.mean(), rel=1e-12)
        assert mom["rms_d"][t] == pytest.approx(dt.std(), rel=1e-12)
        assert mom["n_in_bucket"][t] == oracle.bucket_count(p, zt, dt)
    zt, dt = oracle.track(p, z0, d0, 5)
    assert np.array_equal(z, zt) and np.array_equal(d, dt)


def test_bucket_membership_brute_force_and_edges():
    g = golden_constants()
    for r in (0.0, 0.5):
        p = P(ratio2=r)
        rng = np.random.default_rng(11)
        z = rng.uniform(-1.2, 1.2, 500) * g["z_max"]
        d = rng.uniform(-1.3, 1.3, 500) * g["delta_max"]
        brute = 0
        for zi, di in zip(z, d):
            ph = g["kappa"] * zi
            H = 0.5 * g["eta"] * 6911.5 * di * di + (g["A"] * g["R"] / 4620) * (
                (1 - math.cos(ph)) + 0.5 * r * (1 - math.cos(2 * ph)))
            brute += (abs(zi) < g["z_max"]) and (H < g["H_sep"])
        assert oracle.bucket_count(p, z, d) == brute
        assert oracle.bucket_mask(p, z, d).sum() == brute
    p = P()
    eps = 1e-9
    ez = 1e-6   # H is quadratic in the distance to the unstable fixed point
    z = np.array([0.0, 0.0, g["z_max"] * (1 - ez), g["z_max"] * (1 + ez), 2 * g["z_max"]])
    d = np.array([g["delta_max"] * (1 - eps), g["delta_max"] * (1 + eps), 0.0, 0.0, 0.0])
    assert list(oracle.bucket_mask(p, z, d)) == [True, False, True, False, False]
    assert oracle.bucket_count(p, z[:0], d[:0]) == 0


def test_input_recipe_statistics():
    """The seeded bunches have the structure DESIGN.md states (and SURVEY.md probed)."""
    p = P()
    z, d = wl.make_bunch(wl.CONFIGS[1])
    assert z.size == 100_000
    assert oracle.bucket_count(p, z, d) / z.size == pytest.approx(0.617, abs=5e-3)   # G12
    z, d = wl.make_bunch(wl.CONFIGS[0])
    assert oracle.bucket_count(p, z, d) == z.size == 1000                              # G11
    z, d = wl.gaussian_bunch(100_000, 0.23, 5, truncate=False)
    assert oracle.bucket_count(p, z, d) / z.size == pytest.approx(0.919, abs=5e-3)
    z, d = wl.make_bunch(wl.CONFIGS[4], n=20_000)
    assert oracle.bucket_count(P(ratio2=0.5), z, d) == z.size
    assert wl.matched_sigma_delta(0.23) == pytest.approx(2.0031809091353530e-3, rel=1e-12)
    # reproducible
    z2, d2 = wl.make_bunch(wl.CONFIGS[4], n=20_000)
    assert np.array_equal(z, z2) and np.array_equal(d, d2)
