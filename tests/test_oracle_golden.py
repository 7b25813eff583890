"""The oracle against the numbers the paper prints (tests/golden/paper_printed_values.txt):
the coefficients of the small-T expansions eq. (44)/(45) and the extrapolation weights of eq. (51)."""
import os
from fractions import Fraction

import numpy as np

from oracle import wl_oracle as o

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_printed_values.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = [s.strip() for s in line.split("=")]
            out[k] = float(Fraction(v))
    return out


def test_small_T_integrals_use_the_printed_coefficients():
    g = golden()
    for b, m2, a in ((1.3, 1.0, 0.05), (4.0, 0.5, 0.02), (0.2, 2.0, 0.1)):
        m4, m6 = m2 ** 2, m2 ** 3
        ferm = [g["ferm_T1_b4"] * b ** 4, g["ferm_T2_b4_m2"] * b ** 4 * m2,
                g["ferm_T3_b6"] * b ** 6 + g["ferm_T3_b4_m4"] * b ** 4 * m4,
                g["ferm_T4_b4_m6"] * b ** 4 * m6 + g["ferm_T4_b6_m2"] * b ** 6 * m2]
        scal = [g["scal_T1_b4"] * b ** 4, g["scal_T2_b4_m2"] * b ** 4 * m2,
                g["scal_T3_b4_m4"] * b ** 4 * m4 + g["scal_T3_b6"] * b ** 6,
                g["scal_T4_b6_m2"] * b ** 6 * m2 + g["scal_T4_b4_m6"] * b ** 4 * m6]
        for coef, scalar in ((ferm, False), (scal, True)):
            want = sum(c * a ** (k + 2) / (k + 2) for k, c in enumerate(coef))     # int_0^a c_k T^(k+1) dT
            assert abs(o.small_T_integral(b, m2, a, scalar) / want - 1) < 1e-13


def test_extrapolation_weights_are_the_printed_ones():
    g = golden()
    lev = np.array([[0.7], [1.9], [-0.4]])                        # levels N/4, N/2, N
    W_inf, delta = o.extrapolate(lev)
    want = g["extrap_N"] * lev[2, 0] + g["extrap_N_over_2"] * lev[1, 0] + g["extrap_N_over_4"] * lev[0, 0]
    assert abs(W_inf[0] - want) < 1e-15 and abs(delta[0] - abs(lev[2, 0] - want)) < 1e-15      # eq. (52)
