"""Seeded synthetic bunches and the five BASELINE.json configurations.

This module is the ONE piece shared by the CUDA path's callers (tests, bench.py) and the
oracle's callers: it only *generates inputs*.  It holds none of the tracking arithmetic,
imports neither ``oracle`` nor the CUDA binding, and needs numpy only.

The synthetic bunches stand in for the paper's data files (``data*.csv`` and the
hollow-bunch beam of PAPER.md:74, :80 -- neither is available, the paper states neither
their distribution nor the ring settings).  Shapes and sizes follow the paper's runs
(10^5 x 7*10^4; "usual setting 10^5 to 10^7 macro-particles");
ring, RF and value distributions follow BASELINE.json:configs[0..4].  Recipe and readings
(G11, G12, G19): DESIGN.md "Input recipe".
"""
from __future__ import annotations

import math

import numpy as np

# BASELINE.json:configs[0]: "C=6911.5 m, R=C/2pi, protons with p0=26 GeV/c and gamma=27.7,
# alpha_c=1.92e-3, ... h=4620, V=2.0 MV".  gamma and p0 are taken literally and
# independently (reading G4).
RING = dict(circumference_m=6911.5, gamma=27.7, alpha_c=1.92e-3, p0c_eV=26.0e9,
            charge_e=1.0, harmonic=4620, voltage_V=2.0e6, phi_s=0.0)

# BASELINE.json:configs[i]  (seeds: SURVEY.md sec. 8(d))
CONFIGS = [
    dict(name="cfg0_tiny_gauss", n=1_000, turns=1_000, integrators=("leapfrog",), ratio2=0.0,
         dist="gauss", sigma_z=0.23, seed=16100, mode="fused"),
    dict(name="cfg1_hollow", n=100_000, turns=70_000, integrators=("leapfrog",), ratio2=0.0,
         dist="hollow", seed=16101, mode="fused"),
    dict(name="cfg2_large_gauss", n=1_000_000, turns=100_000, integrators=("leapfrog",),
         ratio2=0.0, dist="gauss", sigma_z=0.35, seed=16102, mode="fused", subsample=10_000),
    dict(name="cfg3_per_turn_moments", n=10_000_000, turns=1_000, integrators=("leapfrog",),
         ratio2=0.0, dist="gauss", sigma_z=0.23, seed=16103, mode="per_turn"),
    dict(name="cfg4_variants", n=1_000_000, turns=10_000,
         integrators=("euler_cromer", "leapfrog", "ruth4"), ratio2=0.5,
         dist="gauss", sigma_z=0.30, seed=16104, mode="fused", subsample=100_000),
]


def ring_numbers(ring: dict = RING, ratio2: float = 0.0) -> dict:
    """Numbers the *input recipe* needs (bucket size, matched momentum spread)."""
    C = ring["circumference_m"]
    g = ring["gamma"]
    h = ring["harmonic"]
    R = C / (2.0 * math.pi)
    beta = math.sqrt(1.0 - 1.0 / g ** 2)
    eta = ring["alpha_c"] - 1.0 / g ** 2
    A = ring.get("charge_e", 1.0) * ring["voltage_V"] / (beta * ring["p0c_eV"])
    K = eta * C * A * h / R
    mu = math.acos(1.0 - 0.5 * K)          # single-harmonic leap-frog tune, always (G19)
    return dict(R=R, beta=beta, eta=eta, A=A, K=K, mu=mu, Qs=mu / (2.0 * math.pi),
                kappa=h / R, z_max=math.pi * R / h, H_sep=2.0 * A * R / h,
                delta_max=2.0 * math.sqrt(A * R / (h * eta * C)), etaC=eta * C, r=ratio2,
                pot_scale=A * R / h)


def matched_sigma_delta(sigma_z: float, ring: dict = RING) -> float:
    """configs[0]: sigma_delta = sigma_z * 2 pi Q_s / (eta C), Q_s = mu / 2 pi (G19)."""
    q = ring_numbers(ring)
    return sigma_z * q["mu"] / q["etaC"]


def _inside_separatrix(z, delta, q):
    """Acceptance test of the input recipe (G11): |z| < z_max and H < H_sep, with the
    Hamiltonian of the RF actually used (including r)."""
    ph = q["kappa"] * z
    pot = (1.0 - np.cos(ph)) + 0.5 * q["r"] * (1.0 - np.cos(2.0 * ph))
    H = 0.5 * q["etaC"] * delta * delta + q["pot_scale"] * pot
    return (np.abs(z) < q["z_max"]) & (H < q["H_sep"])


def gaussian_bunch(n: int, sigma_z: float, seed: int, ring: dict = RING, ratio2: float = 0.0,
                   truncate: bool = True):
    """Gaussian in z and delta (matched sigma_delta), rejection-truncated inside the
    separatrix.  Draw order (G11): per batch, a block of 2n z values then a block of 2n
    delta values from ``default_rng(seed)``; keep the first n accepted pairs in draw order."""
    q = ring_numbers(ring, ratio2)
    sd = matched_sigma_delta(sigma_z, ring)
    rng = np.random.default_rng(seed)
    zs, ds, have = [], [], 0
    batch = max(2 * n, 16)
    while have < n:
        z = rng.normal(0.0, sigma_z, batch)
        d = rng.normal(0.0, sd, batch)
        if truncate:
            m = _inside_separatrix(z, d, q)
            z, d = z[m], d[m]
        zs.append(z)
        ds.append(d)
        have += z.size
    z = np.concatenate(zs)[:n].copy()
    d = np.concatenate(ds)[:n].copy()
    return z, d


def hollow_bunch(n: int, seed: int, ring: dict = RING):
    """configs[1]: in the normalised plane (z, delta*eta*C/(2 pi Q_s)) the radius is uniform
    in [0.4, 0.9]*z_max (linear-uniform) and the phase uniform in [0, 2 pi).  Taken literally
    (G12): no truncation, so part of the ring lies outside the separatrix."""
    q = ring_numbers(ring)
    rng = np.random.default_rng(seed)
    rho = rng.uniform(0.4, 0.9, n) * q["z_max"]
    theta = rng.uniform(0.0, 2.0 * math.pi, n)
    z = rho * np.cos(theta)
    d = rho * np.sin(theta) * q["mu"] / q["etaC"]
    return z, d


def make_bunch(cfg: dict, n: int | None = None, seed: int | None = None, ring: dict = RING):
    """The bunch of one CONFIGS entry (optionally at another size / seed)."""
    n = cfg["n"] if n is None else n
    seed = cfg["seed"] if seed is None else seed
    if cfg["dist"] == "hollow":
        return hollow_bunch(n, seed, ring)
    return gaussian_bunch(n, cfg["sigma_z"], seed, ring, cfg["ratio2"])


def subsample_indices(n: int, m: int, seed: int):
    """Seeded subsample for the oracle (cfg2, cfg4): sorted, without replacement."""
    return np.sort(np.random.default_rng(seed + 1000).choice(n, m, replace=False))


def sigma_delta_for_gate(cfg: dict, ring: dict = RING) -> float:
    """sigma_delta used to normalise |d delta| in the per-particle gate (G17): the matched
    value of the config; cfg1 (hollow) uses cfg0's."""
    return matched_sigma_delta(cfg.get("sigma_z", 0.23), ring)


def shard_range(n: int, rank: int, world: int):
    """Contiguous particle range [lo, hi) of one rank (particles are independent,
    PAPER.md:163): first n % world ranks get one extra particle."""
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


# ---------------------------------------------------------------------------------------------
# Inputs for the rows SURVEY.md sec. 8(f) marks "next" (readings G28-G30).
# Still input generation only: tables, matrices and coordinates are DATA handed to both sides.
# ---------------------------------------------------------------------------------------------
NEXT_CONFIGS = dict(
    # f2: the shape of the paper's profiled hollow-bunch run (10^5 x 7*10^4) with the
    # "parameter changes of the accelerator setting" switched on
    f2_programme=dict(name="f2_programme", n=100_000, turns=70_000, integrator="leapfrog",
                      ratio2=0.0, dist="gauss", sigma_z=0.23, seed=16110, programme_seed=16120),
    # f2 with acceleration ("gamma ramps per turn"; G32): the same
    # run shape, reference momentum 26 -> 60 GeV/c on the synchronous phase (`energy_ramp`)
    f2_ramp=dict(name="f2_ramp", n=100_000, turns=70_000, integrator="leapfrog", ratio2=0.0,
                 dist="gauss", sigma_z=0.08, seed=16113, p_start=26e9, p_end=60e9),
    # f3: "the same matrix is repeatedly acting on the typically 10^5 to 10^7 macro-particles'
    # state vectors"
    f3_transverse=dict(name="f3_transverse", n=1_000_000, turns=10_000, n_seg=4, seed=16111,
                       lattice_seed=16121, sigma_z=0.23, per_turn_n=10_000_000, per_turn_turns=200),
    # f4: slicing at the interaction point every turn, cfg3's shape (10^7 x 10^3)
    f4_slices=dict(name="f4_slices", n=10_000_000, turns=1_000, n_slices=64, dist="gauss",
                   sigma_z=0.23, seed=16112, ratio2=0.0),
)


def ramp_ring_numbers(p0c, ring: dict = RING):
    """A(p) = qV/(beta(p) p) and eta(p) at reference momentum p0c (array or scalar), with the rest
    energy mc2 = p0c_create/(beta gamma) (G32).  Part of the *input recipe* only: it
    places the RF phase programme on the synchronous phase."""
    g = ring["gamma"]
    mc2 = ring["p0c_eV"] / (math.sqrt(1.0 - 1.0 / g ** 2) * g)
    bg = np.asarray(p0c, dtype=np.float64) / mc2
    g2 = 1.0 + bg * bg
    beta = bg / np.sqrt(g2)
    return dict(mc2=mc2, beta=beta, eta=ring["alpha_c"] - 1.0 / g2,
                A=ring.get("charge_e", 1.0) * ring["voltage_V"] / (beta * np.asarray(p0c, dtype=np.float64)))


def energy_ramp(turns: int, p_start: float, p_end: float, ring: dict = RING,
                volt_scale: float = 1.0):
    """f2 with acceleration: (p0c[turns+1], volt_scale[turns], phase_off[turns]).

    The reference momentum goes from p_start to p_end with a rate that starts and ends at zero,
    p(t) = p_start + (p_end - p_start) (t/N - sin(2 pi t/N)/(2 pi)) (a synchrotron's ramp is
    rounded at both ends so that the bunch is not kicked into a dipole oscillation); constant
    voltage; the RF phase programme keeps the reference particle synchronous,
    psi_t = arcsin(D_t / (p0c[t] a_t A(p0c[t]))) (G32).  The paper gives no ramp."""
    t = np.arange(turns + 1, dtype=np.float64)
    N = float(max(turns, 1))
    p0c = p_start + (p_end - p_start) * (t / N - np.sin(2.0 * np.pi * t / N) / (2.0 * np.pi))
    p0c[0], p0c[-1] = p_start, p_end
    a = np.full(turns, float(volt_scale))
    A = ramp_ring_numbers(p0c[:-1], ring)["A"]
    s = np.diff(p0c) / (p0c[:-1] * a * A)
    if np.any(np.abs(s) >= 1.0):
        raise ValueError("ramp too fast for the voltage: |sin(phi_s)| reaches %.3f" % np.abs(s).max())
    return np.ascontiguousarray(p0c), a, np.ascontiguousarray(np.arcsin(s))


def rf_programme(turns: int, seed: int, ring: dict = RING, ramp_to: float = 1.5,
                 mod_amplitude: float = 0.05, mod_tune_ratio: float = 0.95,
                 noise_rms: float = 1e-3):
    """f2 input tables (volt_scale[turns], phase_off[turns]).

    A hollow-bunch style manipulation (the paper gives no numbers for it):
    the voltage ramps linearly from V to ramp_to*V over the run; the RF phase is modulated at
    mod_tune_ratio * Q_s (near-resonant dipole excitation, which is how hollow bunches are
    made) with a half-sine envelope over the first half of the run, plus seeded white RF phase
    noise of noise_rms rad so that no two turns share a table entry."""
    q = ring_numbers(ring)
    t = np.arange(turns, dtype=np.float64)
    a = 1.0 + (ramp_to - 1.0) * t / max(turns - 1, 1)
    half = max(turns // 2, 1)
    env = np.where(t < half, np.sin(np.pi * t / half), 0.0)
    psi = mod_amplitude * env * np.sin(2.0 * np.pi * mod_tune_ratio * q["Qs"] * t)
    psi = psi + np.random.default_rng(seed).normal(0.0, noise_rms, turns)
    return np.ascontiguousarray(a), np.ascontiguousarray(psi)


def twiss_transfer(a1: float, b1: float, a2: float, b2: float, phi: float):
    """Courant-Snyder 2x2 transfer matrix from (alpha1, beta1) to (alpha2, beta2) with phase
    advance phi (textbook form; these are INPUT matrices, not tracking arithmetic)."""
    c, s = math.cos(phi), math.sin(phi)
    r = math.sqrt(b2 / b1)
    return np.array([[r * (c + a1 * s), math.sqrt(b1 * b2) * s],
                     [-((1.0 + a1 * a2) * s + (a2 - a1) * c) / math.sqrt(b1 * b2),
                      (c - a2 * s) / r]])


def transverse_lattice(n_seg: int, seed: int, qx: float = 20.13, qy: float = 20.18,
                       ring: dict = RING, coupling: float = 1e-4):
    """f3 input: n_seg 4x4 segment matrices [n_seg, 4, 4] (row-major) for an SPS-like ring
    (integer tunes 20, BASELINE's circumference).  Segment boundaries carry seeded Twiss
    parameters around the smooth-approximation beta = R/Q; the phase advance is split evenly.
    `coupling` adds a thin skew quadrupole (x' += k y, y' += k x) at the end of every segment so
    that the off-diagonal 2x2 blocks are populated.  Returns (matrices, twiss_at_start) with
    twiss_at_start = (alpha_x, beta_x, alpha_y, beta_y) for matching the bunch."""
    rng = np.random.default_rng(seed)
    R = ring["circumference_m"] / (2.0 * math.pi)
    bx0, by0 = R / qx, R / qy
    ax = rng.uniform(-1.0, 1.0, n_seg)
    ay = rng.uniform(-1.0, 1.0, n_seg)
    bx = bx0 * rng.uniform(0.6, 1.6, n_seg)
    by = by0 * rng.uniform(0.6, 1.6, n_seg)
    mats = np.zeros((n_seg, 4, 4))
    for s in range(n_seg):
        s2 = (s + 1) % n_seg
        m = np.zeros((4, 4))
        m[:2, :2] = twiss_transfer(ax[s], bx[s], ax[s2], bx[s2], 2.0 * math.pi * qx / n_seg)
        m[2:, 2:] = twiss_transfer(ay[s], by[s], ay[s2], by[s2], 2.0 * math.pi * qy / n_seg)
        skew = np.eye(4)
        skew[1, 2] = coupling
        skew[3, 0] = coupling
        mats[s] = skew @ m
    return np.ascontiguousarray(mats), (float(ax[0]), float(bx[0]), float(ay[0]), float(by[0]))


def transverse_bunch(n: int, seed: int, twiss, eps_x: float = 8.0e-8, eps_y: float = 8.0e-8):
    """f3 input: Gaussian (x, x', y, y') matched to `twiss` = (alpha_x, beta_x, alpha_y, beta_y)
    with geometric emittances eps (SPS-like: 2 um normalised at gamma 27.7)."""
    ax, bx, ay, by = twiss
    g = np.random.default_rng(seed).normal(0.0, 1.0, (4, n))
    x = math.sqrt(eps_x * bx) * g[0]
    xp = math.sqrt(eps_x / bx) * (g[1] - ax * g[0])
    y = math.sqrt(eps_y * by) * g[2]
    yp = math.sqrt(eps_y / by) * (g[3] - ay * g[2])
    return tuple(np.ascontiguousarray(v) for v in (x, xp, y, yp))


def slice_grid(cfg: dict, ring: dict = RING):
    """f4 input: the slicing interval = the RF bucket [-z_max, z_max), cfg['n_slices'] slices."""
    q = ring_numbers(ring)
    return -q["z_max"], q["z_max"], int(cfg["n_slices"])
