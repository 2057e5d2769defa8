"""Writes faddeeva_table.h: the coefficient tables of the FP32 device Faddeeva evaluator (me_device.cuh).

Two regions:
  core  |z|^2 <  CUT2 : Weideman (1994) expansion  w(z) = 2 p(Z) D^2 + D / sqrt(pi),
                        D = 1 / (L - i z), Z = (L + i z) D, p a degree N-1 polynomial whose coefficients are the
                        Fourier coefficients of exp(-t^2)(L^2 + t^2) on t = L tan(theta/2), computed here by FFT;
  wing  |z|^2 >= CUT2 : asymptotic series w(z) = (i / sqrt(pi)) s sum_k (2k-1)!! / 2^k  q^k,  s = 1/z, q = s^2.
  far   |z| >= FAR, a <= FAR_AMAX : the same series regrouped.  With s = r (v - i a), r = 1/|z|^2 and v^2 = 1/r - a^2 every term
                        of i s^(2k+1) becomes a polynomial in r and A = a^2:  H = a r X(r; A), F = v r Y(r; A) with X, Y power
                        series in r whose coefficients are polynomials in A (exact rationals, computed here).  On r in
                        [0, 1/T^2] the series (KFAR terms) is cut to degree 3 (T = FAR) or 1 (T = FAR_LIN) by truncating its
                        Chebyshev expansion on that interval (economisation): a linear map of the series coefficients,
                        so the economised coefficients are again polynomials in A, G[j][p] A^p, p <= FAR_PA: the table
                        written here, evaluated once per parameter vector (me_device.cuh far_coef).
Run: python gen_faddeeva_table.py   (numpy only; the header is committed, this script documents its origin; with scipy it
also prints the maximum error of the far tiers against scipy.special.wofz).
"""
import math
import os
from fractions import Fraction

import numpy as np
from numpy.polynomial import chebyshev as cheb
from numpy.polynomial import polynomial as poly

N = 16          # Weideman terms
WL = 3.5        # Weideman's L (his default sqrt(N / sqrt 2) = 3.36 is tuned for the whole line; 3.5 is better on |z| < 5)
K = 5           # highest power of q in the wing series
CUT = 5.0       # region boundary in |z|
FAR = 4.5       # beyond this |z| the far tier (cubics in r = 1/|z|^2 economised from the asymptotic series) is used
FAR_AMAX = 0.75 # largest damping for which the far tier uses the polynomial-in-r form (A r must stay small; me_device.cuh FarCoef)
FAR_LIN = 12.0  # beyond this |z| X, Y are linear in r
W2 = 9.0        # a > FAR_AMAX: beyond this |z| the series itself is cut after q^2, between CUT and W2 after q^K
KFAR = 10       # terms of the asymptotic series that feed the economisation
FAR_PA = 3      # highest power of A = a^2 kept in an economised coefficient


def far_series(kmax):
    """{(i, p): c}: coefficient c (a Fraction, 1/sqrt(pi) left out) of r^i A^p in X and in Y."""
    ck = [Fraction(1)]
    for k in range(1, kmax + 1):
        ck.append(ck[-1] * Fraction(2 * k - 1, 2))
    X, Y = {}, {}
    for k in range(kmax + 1):
        n = 2 * k + 1                                   # i (v - i a)^n r^n
        for m in range(n + 1):
            f = 1j * (-1j) ** m
            if m % 2 == 1:                              # real part: a A^((m-1)/2) (v^2)^((n-m)/2)
                co, j, i, P = int(round(f.real)) * math.comb(n, m), (m - 1) // 2, (n - m) // 2, X
            else:                                       # imaginary part: v A^(m/2) (v^2)^((n-m-1)/2)
                co, j, i, P = int(round(f.imag)) * math.comb(n, m), m // 2, (n - m - 1) // 2, Y
            for t in range(i + 1):                      # (1/r - A)^i = sum_t C(i,t) r^(t-i) (-A)^t, times r^(n-1)
                key = (n - 1 - (i - t), j + t)
                P[key] = P.get(key, 0) + ck[k] * co * math.comb(i, t) * (-1) ** t
    return X, Y


def economise_matrix(n, deg, R):
    """(deg+1) x n: monomial coefficients in r on [0, R] -> those of the Chebyshev expansion on [0, R] cut after T_deg."""
    M = np.zeros((deg + 1, n))
    to_t, to_r = np.array([R / 2, R / 2]), np.array([-1.0, 2.0 / R])       # r(t), t(r)
    for k in range(n):
        pt = poly.polypow(to_t, k)
        cut = cheb.cheb2poly(cheb.poly2cheb(pt)[:deg + 1])
        out = np.zeros(1)
        for i, c in enumerate(cut):
            out = poly.polyadd(out, c * poly.polypow(to_r, i))
        M[:len(out), k] = out
    return M


def far_tables(deg, T):
    """G_X[j][p], G_Y[j][p] (1/sqrt(pi) folded in): coefficient j of the economised X, Y = sum_p G[j][p] A^p."""
    X, Y = far_series(KFAR)
    n = 2 * KFAR + 1
    M = economise_matrix(n, deg, 1.0 / (T * T))
    out = []
    for P in (X, Y):
        G = np.zeros((deg + 1, FAR_PA + 1))
        for (i, p), c in P.items():
            if p <= FAR_PA:
                G[:, p] += M[:, i] * float(c)
        out.append(G / math.sqrt(math.pi))
    return out


def far_error(deg, T, tmax):
    from scipy.special import wofz
    GX, GY = far_tables(deg, T)
    eh = ef = 0.0
    for a in (0.01, 0.05, 0.1, 0.2, 0.3, 0.4, 0.5, 0.6, FAR_AMAX):
        Ap = (a * a) ** np.arange(FAR_PA + 1)
        cx, cy = GX @ Ap, GY @ Ap
        v = np.linspace(math.sqrt(T * T - a * a), tmax, 8000)
        r = 1.0 / (v * v + a * a)
        w = wofz(v + 1j * a)
        eh = max(eh, np.abs(a * r * poly.polyval(r, cx) - w.real).max())
        ef = max(ef, np.abs(v * r * poly.polyval(r, cy) - w.imag).max())
    return eh, ef


def weideman(n):
    m = 2 * n
    k = np.arange(-m + 1, m)
    L = WL
    t = L * np.tan(k * math.pi / m / 2)
    f = np.concatenate([[0.0], np.exp(-t * t) * (L * L + t * t)])
    a = np.real(np.fft.fft(np.fft.fftshift(f))) / (2 * m)
    return L, a[1:n + 1]          # a[0] multiplies Z^0 ... a[n-1] multiplies Z^(n-1)


def lit(x):
    """A C float literal body: always with a decimal point or an exponent."""
    t = "%.9g" % x
    return t if ("." in t or "e" in t) else t + ".0"


def main(path=None):
    """Writes the header (default: faddeeva_table.h beside this script)."""
    L, a = weideman(N)
    c = [1.0 / math.sqrt(math.pi)]
    for k in range(1, K + 1):
        c.append(c[-1] * (2 * k - 1) / 2.0)
    here = os.path.dirname(os.path.abspath(__file__))
    with open(path or os.path.join(here, "faddeeva_table.h"), "w") as fh:
        fh.write("// Generated by gen_faddeeva_table.py — do not edit.\n#pragma once\n")
        fh.write("#define FAD_N %d\n#define FAD_K %d\n" % (N, K))
        fh.write("#define FAD_CUT2 %.2ff\n" % (CUT * CUT))
        fh.write("#define FAD_FAR2 %.1ff\n" % (FAR * FAR))
        fh.write("#define FAD_FAR_AMAX %.2ff\n" % FAR_AMAX)
        # the same boundaries unsquared: tier selection compares dv = min|v| - (outermost Zeeman shift) with them, which
        # guarantees |z| >= boundary for every component of the line
        fh.write("#define FAD_CUT %.1ff\n#define FAD_FAR %.1ff\n#define FAD_FAR_LIN %.1ff\n#define FAD_W2 %.1ff\n" % (CUT, FAR, FAR_LIN, W2))
        # far tiers: economised coefficient j = sum_p G[j][p] A^p, rows j = 0..deg, columns p = 0..FAR_PA
        fh.write("#define FAD_FAR_PA %d\n" % FAR_PA)
        for name, deg, T in (("CUB", 3, FAR), ("LIN", 1, FAR_LIN)):
            for xy, G in zip("XY", far_tables(deg, T)):
                rows = ", ".join("{" + ", ".join("%.9gf" % g for g in row) + "}" for row in G)
                fh.write("#define FAD_%s_%s {%s}\n" % (name, xy, rows))
        fh.write("#define FAD_L %sf\n#define FAD_2L %sf\n" % (lit(L), lit(2 * L)))
        fh.write("#define FAD_INV_SQRTPI %.9gf\n" % (1.0 / math.sqrt(math.pi)))
        for i, x in enumerate(a):
            fh.write("#define FAD_A%d %.9gf\n" % (i, 2.0 * x))          # the factor 2 of 2 p(Z) D^2 is folded in
        for i, x in enumerate(c):
            fh.write("#define FAD_C%d %.9gf\n" % (i, x))
        # Quadratic-factor recurrence over the core coefficients, unrolled: leaves b0, b1 (see me_device.cuh ME_REC).
        fh.write("#define FAD_CORE_RECURRENCE(t, m) \\\n")
        fh.write("    const f2 cb%d = fma2(t, bc(FAD_A%d), FAD_A%d); \\\n" % (N - 2, N - 1, N - 2))
        fh.write("    const f2 cb%d = fma2(t, cb%d, fma2(m, bc(FAD_A%d), FAD_A%d)); \\\n" % (N - 3, N - 2, N - 1, N - 3))
        for k in range(N - 4, -1, -1):
            fh.write("    const f2 cb%d = fma2(t, cb%d, fma2(m, cb%d, FAD_A%d));%s\n" % (k, k + 1, k + 2, k, " \\" if k else ""))


if __name__ == "__main__":
    main()
    try:
        print("far tier, cubic  on |z| >= %.1f: max |dH| %.2e, |dF| %.2e (a <= %.2f, against scipy.special.wofz)" % ((FAR,) + far_error(3, FAR, 14.0) + (FAR_AMAX,)))
        print("far tier, linear on |z| >= %.1f: max |dH| %.2e, |dF| %.2e" % ((FAR_LIN,) + far_error(1, FAR_LIN, 80.0)))
    except ImportError:
        pass
