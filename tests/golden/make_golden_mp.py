"""Writes tests/golden/we1.txt and kepler_values.txt: 40-digit mpmath evaluation of the path's
DEFINITION (steps 1-8; BASELINE.json north_star) for worked
example WE-1 and five Kepler-equation values (SURVEY.md section 8(c) pins P2, P8).

Independent of BOTH implementations: it imports neither oracle/ nor the CUDA package, solves
Kepler's equation by 200 plain Newton steps from E = M at 40 digits, and projects with the VECTOR
form of the gnomonic projection (the oracle uses the trigonometric form).  The paper prints no
worked example (PAPER.md has no numeric orbit/pixel pair), so these are the mathematics' values,
not the paper's.   Run:  python tests/golden/make_golden_mp.py
"""
import os

from mpmath import mp, mpf, sin, cos, sqrt, atan2, asin, pi, floor, radians

mp.dps = 40
HERE = os.path.dirname(os.path.abspath(__file__))
k = mpf("0.01720209895")
GM = k * k
c = mpf("299792.458") * 86400 / mpf("149597870.7")
eps = radians(mpf("23.439281"))
s = radians(mpf("0.2") / 3600)


def kepler(M, e):
    E = M
    for _ in range(200):
        E = E - (E - e * sin(E) - M) / (1 - e * cos(E))
    return E


def helio(el, t, t0):
    a, e, i, Om, w, M0 = el
    n = sqrt(GM / a ** 3)
    M = M0 + n * (t - t0)
    E = kepler(M, e)
    P = (cos(Om) * cos(w) - sin(Om) * sin(w) * cos(i), sin(Om) * cos(w) + cos(Om) * sin(w) * cos(i),
         sin(w) * sin(i))
    Q = (-cos(Om) * sin(w) - sin(Om) * cos(w) * cos(i), -sin(Om) * sin(w) + cos(Om) * cos(w) * cos(i),
         cos(w) * sin(i))
    X = a * (cos(E) - e)
    Y = a * sqrt(1 - e * e) * sin(E)
    return tuple(X * P[j] + Y * Q[j] for j in range(3)), M, E


def chain(el, t, t0, R, ra0, de0, W, H):
    r0, M, E = helio(el, t, t0)
    tau = sqrt(sum((r0[j] - R[j]) ** 2 for j in range(3))) / c
    r1, M1, E1 = helio(el, t - tau, t0)
    d = tuple(r1[j] - R[j] for j in range(3))
    q = (d[0], d[1] * cos(eps) - d[2] * sin(eps), d[1] * sin(eps) + d[2] * cos(eps))
    rho = sqrt(sum(x * x for x in q))
    ra = atan2(q[1], q[0]) % (2 * pi)
    de = asin(q[2] / rho)
    tv = (cos(de0) * cos(ra0), cos(de0) * sin(ra0), sin(de0))
    ee = (-sin(ra0), cos(ra0), mpf(0))
    en = (-sin(de0) * cos(ra0), -sin(de0) * sin(ra0), cos(de0))
    D = sum(q[j] * tv[j] for j in range(3))
    xi = sum(q[j] * ee[j] for j in range(3)) / D
    eta = sum(q[j] * en[j] for j in range(3)) / D
    x = (mpf(W) - 1) / 2 + xi / s
    y = (mpf(H) - 1) / 2 + eta / s
    out = [("M", M), ("E", E), ("r_x", r0[0]), ("r_y", r0[1]), ("r_z", r0[2]), ("tau", tau),
           ("M1", M1), ("E1", E1), ("r1_x", r1[0]), ("r1_y", r1[1]), ("r1_z", r1[2]),
           ("q_x", q[0]), ("q_y", q[1]), ("q_z", q[2]), ("rho", rho), ("ra", ra), ("dec", de),
           ("D", D / rho), ("xi", xi), ("eta", eta), ("x", x), ("y", y),
           ("ix", floor(x + mpf("0.5"))), ("iy", floor(y + mpf("0.5")))]
    return out


def main():
    with open(os.path.join(HERE, "we1.txt"), "w") as f:
        f.write("# WE-1 (SURVEY.md 8(c) P8): a=2.7 e=0.1 i=5deg Omega=80deg omega=30deg M0=250deg t0=0\n"
                "# t=17.25 d, R_obs=(cos kt, sin kt, 0), tangent (6.0288, -0.2457) rad, W=H=256,\n"
                "# constants of DESIGN.md A1.  40-digit mpmath, written by make_golden_mp.py.\n"
                "# D is the direction cosine q.t_hat/|q| (the oracle's trigonometric D).\n")
        f.write("const GM %s\nconst c %s\nconst obliquity %s\nconst pixel_scale %s\n"
                % (mp.nstr(GM, 25), mp.nstr(c, 25), mp.nstr(eps, 25), mp.nstr(s, 25)))
        el = (mpf("2.7"), mpf("0.1"), radians(5), radians(80), radians(30), radians(250))
        t = mpf("17.25")
        R = (cos(k * t), sin(k * t), mpf(0))
        for name, v in chain(el, t, mpf(0), R, mpf("6.0288"), mpf("-0.2457"), 256, 256):
            f.write("%s %s\n" % (name, mp.nstr(v, 25)))
    with open(os.path.join(HERE, "kepler_values.txt"), "w") as f:
        f.write("# e M E  with E - e sin E = M (SURVEY.md 8(c) P2), 40-digit mpmath Newton\n")
        for e, M in [("0.9", "0.05"), ("0.9", "3.0"), ("0.3", "-2.5"), ("0.9", "1e-6"),
                     ("0", "1.234"), ("0.999", "0.001"), ("0.5", "3.141592653589793"),
                     ("0.7", "-0.3"), ("0.2", "2.0"), ("0.95", "6.0")]:
            # values are principal: M is given inside (-pi, pi] except the last, reduced by 2 pi
            Mv = mpf(M)
            Mr = Mv - 2 * pi * floor(Mv / (2 * pi) + mpf("0.5"))
            f.write("%s %s %s\n" % (e, M, mp.nstr(kepler(Mr, mpf(e)), 25)))


if __name__ == "__main__":
    main()
