"""Writes tests/golden/prism_gz_quadrature.txt: reference gz values for single prisms, computed by a route that
never touches the closed form of PAPER.md Eq. 2: numerical quadrature (mpmath, 40 digits) of Newton's law.

    gz = gamma*rho * IIINT z/r^3 dV                                  (z positive down, r from the station)
       = gamma*rho * IINT [ 1/sqrt(x^2+y^2+Z1^2) - 1/sqrt(x^2+y^2+Z2^2) ] dx dy      (z integrated analytically)
       = gamma*rho * INT  [ asinh(x/sqrt(y^2+Z^2)) ]_{x=X1..X2} |_{Z=Z1} - (same)|_{Z=Z2} dy   (x integrated too)

The last line is evaluated by 1-D Gauss-Legendre quadrature for every case; case A is also evaluated from the
2-D line as a cross-check of the reduction.  Uses neither oracle/ nor the CUDA path.  The cases are the ones
listed in SURVEY.md Appendix A.2 (which reports the same 20 digits from its own quadrature).
Run:  python tests/golden/make_quadrature_pins.py
"""
import os

import mpmath as mp

mp.mp.dps = 40
GAMMA = mp.mpf("6.674e-6")   # 6.674e-11 SI * 1e5 -> mGal per (kg/m^3 * m)   (BASELINE.json config 1; reading C4)

# name, station (x,y,z), box (x1,x2,y1,y2,z1,z2), rho
CASES = [
    ("A", (0, 0, 0), (-50, 50, -50, 50, 100, 200), 1000),
    ("B", (130, -70, -1), (0, 50, 0, 50, 0, 50), 500),
    ("C", (25, 25, -1), (0, 50, 0, 50, 0, 50), 1000),
    ("D", (5000, 3000, -1), (0, 100, 0, 100, 1000, 1100), 300),
    ("Dmirror", (5000, 3000, 2101), (0, 100, 0, 100, 1000, 1100), 300),
    ("E", (375, 375, -1), (300, 500, 300, 500, 100, 250), 500),
    ("F", (25, 25, -1), (300, 500, 300, 500, 100, 250), 500),
]


def gz_1d(station, box, rho):
    xo, yo, zo = [mp.mpf(s) for s in station]
    X1, X2, Y1, Y2, Z1, Z2 = [mp.mpf(b) for b in box]
    X1, X2, Y1, Y2, Z1, Z2 = X1 - xo, X2 - xo, Y1 - yo, Y2 - yo, Z1 - zo, Z2 - zo

    def inner(y, Z):
        c = mp.sqrt(y * y + Z * Z)
        return mp.asinh(X2 / c) - mp.asinh(X1 / c)

    # split the y-range at 0 (integrand is smooth but peaked there when Z is small)
    pts = sorted({Y1, Y2} | ({mp.mpf(0)} if Y1 < 0 < Y2 else set()))
    val = mp.quad(lambda y: inner(y, Z1) - inner(y, Z2), pts)
    return GAMMA * rho * val


def gz_2d(station, box, rho):
    xo, yo, zo = [mp.mpf(s) for s in station]
    X1, X2, Y1, Y2, Z1, Z2 = [mp.mpf(b) for b in box]
    X1, X2, Y1, Y2, Z1, Z2 = X1 - xo, X2 - xo, Y1 - yo, Y2 - yo, Z1 - zo, Z2 - zo
    f = lambda x, y: 1 / mp.sqrt(x * x + y * y + Z1 * Z1) - 1 / mp.sqrt(x * x + y * y + Z2 * Z2)
    return GAMMA * rho * mp.quad(f, [X1, 0, X2], [Y1, 0, Y2])


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "prism_gz_quadrature.txt")
    lines = ["# gz (mGal) of one prism at one station by quadrature of Newton's law; NOT from PAPER.md Eq. 2.",
             "# written by tests/golden/make_quadrature_pins.py (mpmath, 40 digits); agrees with SURVEY.md App. A.2.",
             "# gamma = 6.674e-6; columns: name xo yo zo x1 x2 y1 y2 z1 z2 rho gz"]
    for name, st, box, rho in CASES:
        v = gz_1d(st, box, rho)
        if name == "A":
            v2 = gz_2d(st, box, rho)
            assert abs(v - v2) < mp.mpf(10) ** -25 * abs(v), (v, v2)
        lines.append(" ".join([name] + [repr(float(s)) for s in st] + [repr(float(b)) for b in box] +
                              [repr(float(rho)), mp.nstr(v, 22)]))
        print(lines[-1])
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
