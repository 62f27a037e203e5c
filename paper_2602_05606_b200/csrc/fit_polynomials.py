"""Polynomial coefficients of the CUDA math (math_f32.cuh, math_f32x2.cuh, math_f64.cuh).

    python paper_2602_05606_b200/csrc/fit_polynomials.py [f32|f64]

Near-minimax fits by Chebyshev interpolation in 60-digit arithmetic (mpmath): every fitted function is
bounded away from zero on its interval, so absolute and relative error coincide up to a constant.  The
script prints, per function, the degree, the measured maximum relative error on a dense grid and the
coefficients rounded to the target type, ready to paste into the headers.  It belongs to the CUDA path
only: the CPU checker neither imports nor runs it, and nothing here is used at run time.
"""
from __future__ import annotations

import re
import struct
import sys

import mpmath as mp

mp.mp.dps = 60


def cheb_fit(f, lo, hi, deg):
    """Monomial coefficients (ascending, mpf) of the degree-`deg` interpolant of f at the Chebyshev
    nodes of [lo, hi]."""
    n = deg + 1
    lo, hi = mp.mpf(lo), mp.mpf(hi)
    nodes = [mp.cos(mp.pi * (k + mp.mpf(1) / 2) / n) for k in range(n)]
    xs = [(hi - lo) / 2 * t + (hi + lo) / 2 for t in nodes]
    A = mp.matrix(n, n)
    b = mp.matrix(n, 1)
    for i, x in enumerate(xs):
        for j in range(n):
            A[i, j] = x ** j
        b[i] = f(x)
    c = mp.lu_solve(A, b)
    return [c[j] for j in range(n)]


def max_rel_err(f, coefs, lo, hi, rnd, npts=2001):
    """Max relative error of the Horner evaluation with coefficients rounded by `rnd` (exact arithmetic)."""
    cr = [mp.mpf(rnd(c)) for c in coefs]
    worst = mp.mpf(0)
    for k in range(npts):
        x = mp.mpf(lo) + (mp.mpf(hi) - mp.mpf(lo)) * k / (npts - 1)
        p = mp.mpf(0)
        for c in reversed(cr):
            p = p * x + c
        worst = max(worst, abs(p / f(x) - 1))
    return worst


def r32(c):
    return struct.unpack("f", struct.pack("f", float(c)))[0]


def r64(c):
    return float(c)


def hex32(c):
    m = re.match(r"(-?0x1\.)([0-9a-f]*?)0*(p[+-]\d+)$", float.hex(r32(c)))
    return m.group(1) + (m.group(2) or "0") + m.group(3) + "f"


def hex64(c):
    return float.hex(r64(c))


def report(name, f, lo, hi, deg, rnd, fmt):
    c = cheb_fit(f, lo, hi, deg)
    e = max_rel_err(f, c, lo, hi, rnd)
    print("// %s: degree %d on [%s, %s], max relative error %.2e" % (name, deg, lo, hi, float(e)))
    print("//   highest degree first: " + ", ".join(fmt(x) for x in reversed(c)))
    return c


TINY = mp.mpf(10) ** -30


def fits_f32():
    ln2 = mp.log(2)
    report("G(p) = -log2(1-p)/p", lambda p: -mp.log(1 - p) / ln2 / p if p > TINY else 1 / ln2, 0, 0.25, 5, r32, hex32)
    report("R(m) = (2^m - 1)/m", lambda m: (mp.power(2, m) - 1) / m if m > TINY else ln2, 0, 0.5, 4, r32, hex32)
    report("sin(pi q/2)/q in z = q^2", lambda z: mp.sin(mp.pi / 2 * mp.sqrt(z)) / mp.sqrt(z) if z > TINY else mp.pi / 2,
           0, 0.25, 3, r32, hex32)
    report("cos(pi q/2) in z = q^2", lambda z: mp.cos(mp.pi / 2 * mp.sqrt(z)), 0, 0.25, 3, r32, hex32)


def fits_f64():
    # ln(m) = 2 f P(f^2), f = (m-1)/(m+1).  k = round(log2 S) is taken from the high words of numerator and
    # denominator (a piecewise-linear log2, off by < 0.09), so m = S 2^-k lies in [2^-0.59, 2^0.59].
    m = mp.power(2, mp.mpf("0.59"))
    zmax = ((m - 1) / (m + 1)) ** 2
    report("P(z) = atanh(sqrt z)/sqrt z", lambda z: mp.atanh(mp.sqrt(z)) / mp.sqrt(z) if z > TINY else mp.mpf(1),
           0, zmax, 5, r64, hex64)
    # expm1(rho) = rho Q(rho), |rho| <= ln2/2
    h = mp.log(2) / 2 * (1 + mp.mpf(1) / 1000)
    report("Q(rho) = expm1(rho)/rho", lambda r: mp.expm1(r) / r if abs(r) > TINY else mp.mpf(1), -h, h, 8, r64, hex64)
    report("sin(pi q/2)/q in z = q^2", lambda z: mp.sin(mp.pi / 2 * mp.sqrt(z)) / mp.sqrt(z) if z > TINY else mp.pi / 2,
           0, 0.25, 5, r64, hex64)
    report("cos(pi q/2) in z = q^2", lambda z: mp.cos(mp.pi / 2 * mp.sqrt(z)), 0, 0.25, 5, r64, hex64)


if __name__ == "__main__":
    which = sys.argv[1] if len(sys.argv) > 1 else "all"
    if which in ("f32", "all"):
        fits_f32()
    if which in ("f64", "all"):
        fits_f64()
