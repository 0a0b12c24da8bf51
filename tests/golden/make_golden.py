"""Writes tests/golden/*.txt -- expected values for the oracle's pins.

Nothing here calls oracle/ or the CUDA path.  Every number is either a closed form
evaluated with mpmath at 40 digits or the continuous integral of eq 2.8
with the Stokeslet of eq 2.9 (sign/identity per DESIGN.md reading A1)
computed by adaptive Gauss-Legendre quadrature (mpmath.quad) -- i.e. the mathematics the
trapezoid rule of PAPER.md:173 converges to spectrally fast for far targets.

Run:  python tests/golden/make_golden.py
"""
import os

import mpmath as mp

mp.mp.dps = 40
HERE = os.path.dirname(os.path.abspath(__file__))


def stokeslet_apply(rx, ry, gx, gy):
    """4 pi mu G(r) g  with  G = (-log|r| I + r r^T/|r|^2)/(4 pi mu)."""
    r2 = rx * rx + ry * ry
    ml = -mp.log(r2) / 2
    d = (rx * gx + ry * gy) / r2
    return ml * gx + d * rx, ml * gy + d * ry


def point_stokeslet_cases():
    # one source at the origin with g = (0.3, -0.7); targets chosen so each term is visible
    g = (mp.mpf("0.3"), mp.mpf("-0.7"))
    targets = [(mp.mpf(1), mp.mpf(0)),                       # log term vanishes: 4piU = (gx, 0)
               (mp.e, mp.mpf(0)),                            # -log = -1: 4piU = (0, -gy)... see file
               (2 * mp.cos(mp.mpf("0.7")), 2 * mp.sin(mp.mpf("0.7"))),
               (mp.mpf("-0.25"), mp.mpf("1.5"))]
    rows = []
    for (x, y) in targets:
        ux, uy = stokeslet_apply(x, y, g[0], g[1])
        rows.append((x, y, g[0], g[1], ux, uy))
    return rows


def ellipse(a, b, al):
    return a * mp.cos(al), b * mp.sin(al)


def sli_continuous(shape, density, target):
    """4 pi mu S[f](x) = int_0^{2pi} (4 pi mu G)(x - X(al)) f(al) |X'(al)| dal by mpmath.quad."""
    def integrand(comp):
        def f(al):
            X, Y, dX, dY = shape(al)
            fx, fy = density(al)
            sa = mp.sqrt(dX * dX + dY * dY)
            u = stokeslet_apply(target[0] - X, target[1] - Y, fx * sa, fy * sa)
            return u[comp]
        return f
    pts = [mp.mpf(k) * mp.pi / 8 for k in range(17)]
    return mp.quad(integrand(0), pts), mp.quad(integrand(1), pts)


def main():
    fmt = lambda v: mp.nstr(v, 25)

    with open(os.path.join(HERE, "point_stokeslet.txt"), "w") as fh:
        fh.write("# Closed form of ONE point Stokeslet, eq 2.9 (PAPER.md:133-136; -log|r| I + r r^T/|r|^2, reading A1).\n")
        fh.write("# source at origin, mu = 1.  columns: x y gx gy  4*pi*U_x  4*pi*U_y   (mpmath, 40 digits)\n")
        for row in point_stokeslet_cases():
            fh.write(" ".join(fmt(v) for v in row) + "\n")

    # constant density e on a circle of radius R: closed form AND independent quadrature
    R = mp.mpf("0.8")
    e = (mp.mpf("0.6"), mp.mpf("-0.8"))
    circ = lambda al: (R * mp.cos(al), R * mp.sin(al), -R * mp.sin(al), R * mp.cos(al))
    with open(os.path.join(HERE, "circle_constant_density.txt"), "w") as fh:
        fh.write("# 4*pi*mu*S[e](x) for constant density e on a circle radius R centred at the origin (eq 2.8/2.9).\n")
        fh.write("# closed form (multipole expansion of log|x-y|, |x| = rho >= R):\n")
        fh.write("#   -2 pi R ln(rho) e + 2 pi R x (x.e)/rho^2 + pi R^3 ( e/rho^2 - 2 x (x.e)/rho^4 )\n")
        fh.write("# columns: R ex ey x y  closed_x closed_y  quad_x quad_y   (quad = mpmath.quad of the integral)\n")
        for (x, y) in [(mp.mpf("1.7"), mp.mpf("0.4")), (mp.mpf("-2.0"), mp.mpf("2.5")), (mp.mpf("0.3"), mp.mpf("-3.1"))]:
            rho2 = x * x + y * y
            xe = x * e[0] + y * e[1]
            cf = []
            for comp, (xc, ec) in enumerate(((x, e[0]), (y, e[1]))):
                cf.append(-2 * mp.pi * R * mp.log(rho2) / 2 * ec + 2 * mp.pi * R * xc * xe / rho2
                          + mp.pi * R ** 3 * (ec / rho2 - 2 * xc * xe / rho2 ** 2))
            q = sli_continuous(circ, lambda al: e, (x, y))
            assert abs(cf[0] - q[0]) < mp.mpf("1e-25") and abs(cf[1] - q[1]) < mp.mpf("1e-25"), (cf, q)
            fh.write(" ".join(fmt(v) for v in (R, e[0], e[1], x, y, cf[0], cf[1], q[0], q[1])) + "\n")

    # general smooth density on the ellipse (1, 0.4), rotated/translated: continuous integral
    a, b = mp.mpf(1), mp.mpf("0.4")
    th = mp.mpf("0.35")
    c0 = (mp.mpf("0.2"), mp.mpf("-0.1"))
    ct, st = mp.cos(th), mp.sin(th)

    def ell(al):
        X0, Y0 = a * mp.cos(al), b * mp.sin(al)
        dX0, dY0 = -a * mp.sin(al), b * mp.cos(al)
        return (c0[0] + ct * X0 - st * Y0, c0[1] + st * X0 + ct * Y0,
                ct * dX0 - st * dY0, st * dX0 + ct * dY0)

    dens = lambda al: (mp.mpf("0.5") + mp.cos(2 * al) - mp.mpf("0.3") * mp.sin(al),
                       mp.mpf("-0.2") + mp.mpf("0.7") * mp.sin(3 * al) + mp.mpf("0.4") * mp.cos(al))
    with open(os.path.join(HERE, "ellipse_smooth_density.txt"), "w") as fh:
        fh.write("# 4*pi*mu*S[f](x), continuous integral of eq 2.8 with eq 2.9 by mpmath.quad (40 digits).\n")
        fh.write("# ellipse semi-axes (1, 0.4), rotated by 0.35 rad, centre (0.2,-0.1), X(al) = c + R(th)(a cos al, b sin al)\n")
        fh.write("# density f(al) = (0.5 + cos 2al - 0.3 sin al,  -0.2 + 0.7 sin 3al + 0.4 cos al)\n")
        fh.write("# columns: x y  4piS_x 4piS_y\n")
        for (x, y) in [(mp.mpf("2.4"), mp.mpf("0.3")), (mp.mpf("-1.1"), mp.mpf("2.2")), (mp.mpf("0.4"), mp.mpf("-2.6")),
                       (mp.mpf("3.0"), mp.mpf("3.0"))]:
            q = sli_continuous(ell, dens, (x, y))
            fh.write(" ".join(fmt(v) for v in (x, y, q[0], q[1])) + "\n")

    # perimeter of the ellipse (1, 0.4): 4 a E(m), m = 1 - b^2/a^2
    with open(os.path.join(HERE, "ellipse_perimeter.txt"), "w") as fh:
        fh.write("# perimeter of the ellipse with semi-axes (1, 0.4): 4 a E(1 - b^2/a^2), complete elliptic integral (mpmath.ellipe)\n")
        fh.write(fmt(4 * a * mp.ellipe(1 - b * b / (a * a))) + "\n")


if __name__ == "__main__":
    main()
