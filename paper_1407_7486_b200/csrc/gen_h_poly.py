"""Prints the polynomial coefficients used by wl_field_device.cuh (CUDA path only).

h(u) = [u tanh u - ln cosh u]/u^2 is even and analytic in w = u^2 for |w| < pi^2/4, so near
the axis the kernels evaluate a polynomial in w instead of the closed form, whose
subtraction loses digits as u -> 0.  This script interpolates h at
Chebyshev nodes of [0, w_max] with mpmath (50 digits), converts to monomial coefficients
in w and reports the maximum relative error on a fine grid.

Usage:  python gen_h_poly.py <w_max> <degree>          h(w) on [0, w_max]
        python gen_h_poly.py L <degree>                1 - log2(1+E) on E in [0, 1] (absolute error)
        python gen_h_poly.py Lw <w_min> <degree>       the same on E in [0, 1.001 * 2^-sqrt(w_min)]: the range of E = 2^(-u') when
                                                       u'^2 >= w_min (the "far block" tiers of wl_terms_packed_f32.cuh)
        python gen_h_poly.py E2 <degree>               2^(-f) on f in [-1/2, 1/2] (relative error)
        python gen_h_poly.py hs <w_max> <degree>       h rescaled for the packed FP32 / lean FP64 kernels:
                                                       h(w)/(4 log2 e) as a polynomial in w' = 4 (log2 e)^2 w
Not imported by anything; the printed numbers were pasted into wl_field_device.cuh.
Independent of oracle/ (which uses the Maclaurin series for u < 0.1).
"""
import sys

import mpmath as mp

mp.mp.dps = 50


def h(w):
    w = mp.mpf(w)
    if w == 0:
        return mp.mpf(1) / 2
    u = mp.sqrt(w)
    return (u * mp.tanh(u) - mp.log(mp.cosh(u))) / w


def fit(w_max, deg, f=h, lo=0):
    n = deg + 1
    nodes = [(mp.cos(mp.pi * (2 * k + 1) / (2 * n)) + 1) / 2 * (w_max - lo) + lo for k in range(n)]
    A = mp.matrix(n, n)
    b = mp.matrix(n, 1)
    for r, x in enumerate(nodes):
        for c in range(n):
            A[r, c] = x ** c
        b[r] = f(x)
    coef = mp.lu_solve(A, b)
    return [coef[i] for i in range(n)]


def L(E):
    return 1 - mp.log(1 + mp.mpf(E), 2)


def max_abs_err(coef, x_max, f, cast):
    worst = mp.mpf(0)
    for k in range(2001):
        x = mp.mpf(x_max) * k / 2000
        acc = mp.mpf(0)
        for c in reversed(coef):
            acc = acc * x + cast(c)
        worst = max(worst, abs(acc - f(x)))
    return worst


def max_rel_err(coef, w_max, cast):
    worst = mp.mpf(0)
    for k in range(2001):
        w = mp.mpf(w_max) * k / 2000
        acc = mp.mpf(0)
        for c in reversed(coef):
            acc = acc * w + cast(c)
        worst = max(worst, abs(acc / h(w) - 1))
    return worst


def f32(c):
    import struct
    return mp.mpf(struct.unpack("f", struct.pack("f", float(c)))[0])


if __name__ == "__main__":
    if sys.argv[1] == "L":
        deg = int(sys.argv[2])
        coef = fit(1, deg, L)
        print("// 1 - log2(1+E), E in [0, 1], degree %d" % deg)
        print("// max abs. error: exact coefficients %s, float32 coefficients %s"
              % (mp.nstr(max_abs_err(coef, 1, L, lambda c: c), 3), mp.nstr(max_abs_err(coef, 1, L, f32), 3)))
        for i, c in enumerate(coef):
            print("c%d = %s" % (i, mp.nstr(c, 20)))
        sys.exit(0)
    if sys.argv[1] == "Lw":
        w_min, deg = float(sys.argv[2]), int(sys.argv[3])
        e_max = mp.power(2, -mp.sqrt(w_min)) * mp.mpf("1.001")
        coef = fit(e_max, deg, L)
        print("// 1 - log2(1+E), E in [0, %s] (u'^2 >= %g), degree %d" % (mp.nstr(e_max, 8), w_min, deg))
        print("// max abs. error: exact coefficients %s, float32 coefficients %s"
              % (mp.nstr(max_abs_err(coef, e_max, L, lambda c: c), 3), mp.nstr(max_abs_err(coef, e_max, L, f32), 3)))
        print("{ " + ", ".join("%sf" % mp.nstr(c, 12) for c in coef) + " }")
        sys.exit(0)
    if sys.argv[1] == "E2":
        deg = int(sys.argv[2])
        f = lambda x: mp.power(2, -x)
        coef = fit(mp.mpf(1) / 2, deg, f, lo=-mp.mpf(1) / 2)
        worst = mp.mpf(0)
        for k in range(2001):
            x = -mp.mpf(1) / 2 + mp.mpf(k) / 2000
            acc = mp.mpf(0)
            for c in reversed(coef):
                acc = acc * x + c
            worst = max(worst, abs(acc / f(x) - 1))
        print("// 2^(-f), f in [-1/2, 1/2], degree %d, max rel. error %s" % (deg, mp.nstr(worst, 3)))
        for i, c in enumerate(coef):
            print("c%d = %s" % (i, mp.nstr(c, 20)))
        sys.exit(0)
    if sys.argv[1] == "hs":
        w_max, deg = float(sys.argv[2]), int(sys.argv[3])
        coef = fit(w_max, deg)
        l2e = 1 / mp.log(2)
        k2 = 4 * l2e * l2e
        sc = [c / (4 * l2e) / k2 ** i for i, c in enumerate(coef)]
        print("// h(w)/(4 log2 e) in w' = 4 (log2 e)^2 w, w in [0, %g] (w' < %s), degree %d" % (w_max, mp.nstr(w_max * k2, 10), deg))
        print("// max rel. error of h: exact coefficients %s, float32 coefficients %s"
              % (mp.nstr(max_rel_err(coef, w_max, lambda c: c), 3), mp.nstr(max_rel_err(coef, w_max, f32), 3)))
        for i, c in enumerate(sc):
            print("c%d = %s" % (i, mp.nstr(c, 20)))
        sys.exit(0)
    w_max = float(sys.argv[1])
    deg = int(sys.argv[2])
    coef = fit(w_max, deg)
    print("// h(w), w = u^2 in [0, %g], degree %d" % (w_max, deg))
    print("// max rel. error (exact coefficients): %s" % mp.nstr(max_rel_err(coef, w_max, lambda c: c), 3))
    for i, c in enumerate(coef):
        print("c%d = %s" % (i, mp.nstr(c, 20)))
