"""Writes tests/golden/hand_values.txt, tests/golden/phi_s_values.txt and
tests/golden/derived_constants.txt.

Independent of BOTH implementations: it imports neither ``oracle`` nor the CUDA binding,
only mpmath, and iterates the map of BASELINE.json:configs[0] / configs[4] by hand in
40-digit decimal arithmetic ("Tiny ensembles must match hand-iterated values",
BASELINE.json:north_star (3)).  The same numbers are printed in SURVEY.md sec. 8(c),
"What pins the oracle", item 5 and the table at the top of sec. 8; this script is how
they can be regenerated and checked.

    One turn (configs[0]):  z -= eta*C/2*delta; delta += A*sin(h*z/R); z -= eta*C/2*delta
    Kick (configs[4]):      delta += A*[sin(h*z/R) + r*sin(2h*z/R)]
    Euler-Cromer (G8):      delta += F(z); z -= eta*C*delta
    Ruth4 (G9):             leap-frog steps with factors x1, x0, x1,
                            x1 = 1/(2-2^(1/3)), x0 = -2^(1/3)/(2-2^(1/3))
    Synchronous phase (G3): F(z) = A*[sin(phi_s + h*z/R) - sin(phi_s) + r*sin(2h*z/R)]
                            (phi_s_values.txt: phi_s = 0.3 and -0.7, r = 0 and 0.25; pins the
                            sign of phi_s, the subtracted sin(phi_s) and that the harmonic at 2h
                            carries no phi_s -- none of which the linear tune can see)

Run:  python tests/golden/make_hand_values.py
"""
import os

from mpmath import acos, cbrt, mp, mpf, nstr, pi, sin, sqrt

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
K = eta * C * A * h / R
mu = acos(1 - K / 2)
w = cbrt(2)
x1 = 1 / (2 - w)
x0 = -w / (2 - w)


def kick(z, r, phi_s=0):
    return A * (sin(phi_s + kappa * z) - sin(phi_s) + r * sin(2 * kappa * z))


def leapfrog(z, dl, r, tau=1, phi_s=0):
    z = z - tau * d * dl
    dl = dl + tau * kick(z, r, phi_s)
    z = z - tau * d * dl
    return z, dl


def euler_cromer(z, dl, r, phi_s=0):
    dl = dl + kick(z, r, phi_s)
    z = z - 2 * d * dl
    return z, dl


def ruth4(z, dl, r, phi_s=0):
    for tau in (x1, x0, x1):
        z, dl = leapfrog(z, dl, r, tau, phi_s)
    return z, dl


MAPS = (("leapfrog", leapfrog), ("euler_cromer", euler_cromer), ("ruth4", ruth4))
STARTS = (("0.1", "0"), ("0.5", "-1e-3"), ("-0.7", "5e-4"), ("0", "5e-3"))
PHI_S = ("0.3", "-0.7")
PHI_S_RATIOS = ("0", "0.25")


def main():
    with open(os.path.join(HERE, "derived_constants.txt"), "w") as f:
        f.write("# 40-digit values of the derived constants of BASELINE.json:configs[0]'s ring\n"
                "# (SURVEY.md sec. 8 table). Written by make_hand_values.py (mpmath only).\n"
                "# name value\n")
        for name, val in (("R", R), ("beta", beta), ("eta", eta), ("A", A), ("d", d),
                          ("kappa", kappa), ("K", K), ("mu", mu), ("Qs", mu / (2 * pi)),
                          ("z_max", pi * R / h), ("H_sep", 2 * A * R / h),
                          ("delta_max", 2 * sqrt(A * R / (h * eta * C))),
                          ("x1", x1), ("x0", x0)):
            f.write("%s %s\n" % (name, nstr(val, 25)))
    with open(os.path.join(HERE, "hand_values.txt"), "w") as f:
        f.write("# Hand-iterated (40-digit mpmath) values of the map of BASELINE.json:configs[0]\n"
                "# and configs[4]; same numbers as SURVEY.md sec. 8(c) item 5.\n"
                "# Written by make_hand_values.py (mpmath only, no oracle, no CUDA).\n"
                "# integrator r z0 delta0 turns z delta\n")
        for name, fn in MAPS:
            for r in ("0", "0.5"):
                for z0, d0 in STARTS:
                    z, dl = mpf(z0), mpf(d0)
                    for t in range(1, 1001):
                        z, dl = fn(z, dl, mpf(r))
                        if t in (1, 3, 1000):
                            f.write("%s %s %s %s %d %s %s\n"
                                    % (name, r, z0, d0, t, nstr(z, 22), nstr(dl, 22)))
    with open(os.path.join(HERE, "phi_s_values.txt"), "w") as f:
        f.write("# Hand-iterated (40-digit mpmath) values of the map with a synchronous phase,\n"
                "# F(z) = A [sin(phi_s + kappa z) - sin(phi_s) + r sin(2 kappa z)]  (DESIGN.md G3).\n"
                "# Written by make_hand_values.py (mpmath only, no oracle, no CUDA).\n"
                "# integrator phi_s r z0 delta0 turns z delta\n")
        for name, fn in MAPS:
            for phi in PHI_S:
                for r in PHI_S_RATIOS:
                    for z0, d0 in STARTS:
                        z, dl = mpf(z0), mpf(d0)
                        for t in range(1, 1001):
                            z, dl = fn(z, dl, mpf(r), phi_s=mpf(phi))
                            if t in (1, 3, 1000):
                                f.write("%s %s %s %s %s %d %s %s\n"
                                        % (name, phi, r, z0, d0, t, nstr(z, 22), nstr(dl, 22)))


if __name__ == "__main__":
    main()
