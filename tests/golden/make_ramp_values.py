"""Writes tests/golden/ramp_values.txt: hand-iterated (40-digit mpmath) values of the map with an
energy ramp ("gamma ramps per turn"; reading G32 of DESIGN.md):

    reference momentum p0c[t] -> p0c[t+1] over turn t+1;  mc2 = p0c_create / (beta gamma)
    beta(p), eta(p) from bg = p / mc2;  A(p) = V / (beta(p) p);  d(p) = eta(p) C / 2
    sub-step(tau, pb -> pa):
        z     -= tau d(pb) delta
        delta  = (delta + tau a_t A(pb) [sin(kappa z + psi_t) + r sin(2 (kappa z + psi_t))]
                  - (pa - pb)/pb) * (pb / pa)
        z     -= tau d(pa) delta
    leap-frog = sub-step(1, pb, pa);  Euler-Cromer = kick line, then z -= 2 d(pa) delta;
    Ruth4 = sub-steps (x1, x0, x1) over pb -> pb + x1 D -> (that) + x0 D -> pa,  D = pa - pb.

Independent of BOTH implementations: imports neither ``oracle`` nor the CUDA binding, only
mpmath.  Ring and start points as in make_hand_values.py (BASELINE.json:configs[0], [4]).

Run:  python tests/golden/make_ramp_values.py
"""
import os

from mpmath import cbrt, mp, mpf, nstr, pi, sin, sqrt

mp.dps = 40
HERE = os.path.dirname(os.path.abspath(__file__))

C = mpf("6911.5")
gamma0 = mpf("27.7")
alpha_c = mpf("1.92e-3")
h = 4620
p0c_create = mpf("26e9")
V = mpf("2.0e6")

R = C / (2 * pi)
kappa = h / R
mc2 = p0c_create / (sqrt(1 - 1 / gamma0 ** 2) * gamma0)
w = cbrt(2)
x1 = 1 / (2 - w)
x0 = -w / (2 - w)

# decimal strings, so that mpmath and the tests read the same numbers.  A violent ramp (up, down,
# flat, up) so that every term matters in the leading digits.
P0C = ("26e9", "26.4e9", "27.1e9", "26.9e9", "26.9e9", "28.0e9")
VOLT_SCALE = ("1.0", "0.5", "1.25", "0.0", "2.0")
PHASE_OFF = ("0.2", "0.3", "-0.2", "1.0", "-1.5")
STARTS = (("0.1", "0"), ("0.5", "-1e-3"), ("-0.7", "5e-4"), ("0", "5e-3"))


def ring_at(p):
    bg = p / mc2
    g2 = 1 + bg * bg
    beta = bg / sqrt(g2)
    eta = alpha_c - 1 / g2
    return V / (beta * p), eta * C / 2          # A(p), d(p)


def kick(z, dl, r, a, psi, tau, pb, pa):
    A, _ = ring_at(pb)
    ph = kappa * z + psi
    dl = dl + tau * a * A * (sin(ph) + r * sin(2 * ph)) - (pa - pb) / pb
    return dl * pb / pa


def substep(z, dl, r, a, psi, tau, pb, pa):
    z = z - tau * ring_at(pb)[1] * dl
    dl = kick(z, dl, r, a, psi, tau, pb, pa)
    z = z - tau * ring_at(pa)[1] * dl
    return z, dl


def leapfrog(z, dl, r, a, psi, pb, pa):
    return substep(z, dl, r, a, psi, 1, pb, pa)


def euler_cromer(z, dl, r, a, psi, pb, pa):
    dl = kick(z, dl, r, a, psi, 1, pb, pa)
    z = z - 2 * ring_at(pa)[1] * dl
    return z, dl


def ruth4(z, dl, r, a, psi, pb, pa):
    D = pa - pb
    p1 = pb + x1 * D
    p2 = p1 + x0 * D
    z, dl = substep(z, dl, r, a, psi, x1, pb, p1)
    z, dl = substep(z, dl, r, a, psi, x0, p1, p2)
    return substep(z, dl, r, a, psi, x1, p2, pa)


MAPS = (("leapfrog", leapfrog), ("euler_cromer", euler_cromer), ("ruth4", ruth4))


def main():
    with open(os.path.join(HERE, "ramp_values.txt"), "w") as f:
        f.write("# Hand-iterated (40-digit mpmath) values of the map with an energy ramp\n"
                "# p0c        = %s\n# volt_scale = %s\n# phase_off  = %s\n"
                "# (p0c[t] -> p0c[t+1] over turn t+1; DESIGN.md G32).\n"
                "# Written by make_ramp_values.py (mpmath only, no oracle, no CUDA).\n"
                "# integrator r z0 delta0 turns z delta\n"
                % (" ".join(P0C), " ".join(VOLT_SCALE), " ".join(PHASE_OFF)))
        A0, d0_ = ring_at(p0c_create)
        f.write("# mc2 = %s  A(26e9) = %s  d(26e9) = %s  A(28e9) = %s  d(28e9) = %s\n"
                % (nstr(mc2, 22), nstr(A0, 22), nstr(d0_, 22), nstr(ring_at(mpf("28e9"))[0], 22),
                   nstr(ring_at(mpf("28e9"))[1], 22)))
        for name, fn in MAPS:
            for r in ("0", "0.5"):
                for z0, d0 in STARTS:
                    z, dl = mpf(z0), mpf(d0)
                    for t in range(len(VOLT_SCALE)):
                        z, dl = fn(z, dl, mpf(r), mpf(VOLT_SCALE[t]), mpf(PHASE_OFF[t]),
                                   mpf(P0C[t]), mpf(P0C[t + 1]))
                        if t + 1 in (1, 2, 3, 5):
                            f.write("%s %s %s %s %d %s %s\n"
                                    % (name, r, z0, d0, t + 1, nstr(z, 22), nstr(dl, 22)))


if __name__ == "__main__":
    main()
