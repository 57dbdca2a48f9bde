"""Writes tests/golden/programme_values.txt (phi_s = 0) and
tests/golden/programme_phi_s_values.txt (phi_s = 0.3, -0.7; r = 0, 0.25): hand-iterated (40-digit mpmath) values of the map
with a turn-dependent RF programme (reading G28 of DESIGN.md):

    programme entry t = (a_t, psi_t) applies to every kick of turn t+1,
    F_t(z) = a_t A [ sin(phi_s + kappa z + psi_t) - sin(phi_s) + r sin(2 (kappa z + psi_t)) ]

Independent of BOTH implementations: imports neither ``oracle`` nor the CUDA binding, only
mpmath.  Ring, integrators and start points as in make_hand_values.py
(BASELINE.json:configs[0], configs[4]).

Run:  python tests/golden/make_programme_values.py
"""
import os

from mpmath import cbrt, mp, mpf, nstr, pi, sin, sqrt

mp.dps = 40
HERE = os.path.dirname(os.path.abspath(__file__))

C = mpf("6911.5")
gamma = mpf("27.7")
alpha_c = mpf("1.92e-3")
h = 4620
p0c = mpf("26e9")
V = mpf("2.0e6")

R = C / (2 * pi)
beta = sqrt(1 - 1 / gamma ** 2)
eta = alpha_c - 1 / gamma ** 2
A = V / (beta * p0c)
d = eta * C / 2
kappa = h / R
w = cbrt(2)
x1 = 1 / (2 - w)
x0 = -w / (2 - w)

# the programme: decimal strings, so that both mpmath and the tests read the same numbers
VOLT_SCALE = ("1.0", "0.5", "1.25", "0.0", "2.0")
PHASE_OFF = ("0.0", "0.3", "-0.2", "1.0", "-1.5")
STARTS = (("0.1", "0"), ("0.5", "-1e-3"), ("-0.7", "5e-4"), ("0", "5e-3"))


def kick(z, r, a, psi, phi_s=0):
    ph = kappa * z + psi
    return a * A * (sin(phi_s + ph) - sin(phi_s) + r * sin(2 * ph))


def leapfrog(z, dl, r, a, psi, tau=1, phi_s=0):
    z = z - tau * d * dl
    dl = dl + tau * kick(z, r, a, psi, phi_s)
    z = z - tau * d * dl
    return z, dl


def euler_cromer(z, dl, r, a, psi, phi_s=0):
    dl = dl + kick(z, r, a, psi, phi_s)
    z = z - 2 * d * dl
    return z, dl


def ruth4(z, dl, r, a, psi, phi_s=0):
    for tau in (x1, x0, x1):
        z, dl = leapfrog(z, dl, r, a, psi, tau, phi_s)
    return z, dl


MAPS = (("leapfrog", leapfrog), ("euler_cromer", euler_cromer), ("ruth4", ruth4))
PHI_S = ("0.3", "-0.7")
PHI_S_RATIOS = ("0", "0.25")


def main():
    with open(os.path.join(HERE, "programme_values.txt"), "w") as f:
        f.write("# Hand-iterated (40-digit mpmath) values of the map with the RF programme\n"
                "# volt_scale = %s\n# phase_off  = %s\n"
                "# (entry t applies to every kick of turn t+1; DESIGN.md G28).\n"
                "# Written by make_programme_values.py (mpmath only, no oracle, no CUDA).\n"
                "# integrator r z0 delta0 turns z delta\n"
                % (" ".join(VOLT_SCALE), " ".join(PHASE_OFF)))
        for name, fn in MAPS:
            for r in ("0", "0.5"):
                for z0, d0 in STARTS:
                    z, dl = mpf(z0), mpf(d0)
                    for t in range(len(VOLT_SCALE)):
                        z, dl = fn(z, dl, mpf(r), mpf(VOLT_SCALE[t]), mpf(PHASE_OFF[t]))
                        if t + 1 in (1, 2, 3, 5):
                            f.write("%s %s %s %s %d %s %s\n"
                                    % (name, r, z0, d0, t + 1, nstr(z, 22), nstr(dl, 22)))
    with open(os.path.join(HERE, "programme_phi_s_values.txt"), "w") as f:
        f.write("# Hand-iterated (40-digit mpmath) values of the map with the RF programme\n"
                "# volt_scale = %s\n# phase_off  = %s\n"
                "# and a synchronous phase: F_t(z) = a_t A [sin(phi_s + kappa z + psi_t) - sin(phi_s)\n"
                "# + r sin(2 (kappa z + psi_t))]  (DESIGN.md G3, G28: sin(phi_s) is scaled by a_t, not\n"
                "# shifted by psi_t; the 2h term carries 2 psi_t and no phi_s).\n"
                "# Written by make_programme_values.py (mpmath only, no oracle, no CUDA).\n"
                "# integrator phi_s r z0 delta0 turns z delta\n"
                % (" ".join(VOLT_SCALE), " ".join(PHASE_OFF)))
        for name, fn in MAPS:
            for phi in PHI_S:
                for r in PHI_S_RATIOS:
                    for z0, d0 in STARTS:
                        z, dl = mpf(z0), mpf(d0)
                        for t in range(len(VOLT_SCALE)):
                            z, dl = fn(z, dl, mpf(r), mpf(VOLT_SCALE[t]), mpf(PHASE_OFF[t]),
                                       phi_s=mpf(phi))
                            if t + 1 in (1, 2, 3, 5):
                                f.write("%s %s %s %s %s %d %s %s\n"
                                        % (name, phi, r, z0, d0, t + 1, nstr(z, 22), nstr(dl, 22)))


if __name__ == "__main__":
    main()
