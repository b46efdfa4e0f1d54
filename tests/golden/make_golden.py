"""Writes tests/golden/chang_refsdal_cusps.txt from the closed forms (no oracle, no CUDA).

Cusps of the Chang-Refsdal caustic of one unit-mass star at the origin (Eq. 12 and
:128 Eq. 15 with N = 1): real-axis cusps at +-2 gamma / sqrt(1 - kappa_s - gamma) (phi = 0) and
imaginary-axis cusps at +-2 gamma / sqrt(1 - kappa_s + gamma) (phi = pi).
"""
import os
from decimal import Decimal, getcontext

getcontext().prec = 40
CASES = [("0.2", "0.35"), ("0.0", "0.3"), ("0.0", "0.4"), ("0.1", "0.1")]

here = os.path.dirname(os.path.abspath(__file__))
with open(os.path.join(here, "chang_refsdal_cusps.txt"), "w") as f:
    f.write("# kappa_s gamma real_axis_cusp(phi=0) imag_axis_cusp(phi=pi)\n")
    for ks, g in CASES:
        ks_d, g_d = Decimal(ks), Decimal(g)
        re = 2 * g_d / (1 - ks_d - g_d).sqrt()
        im = 2 * g_d / (1 - ks_d + g_d).sqrt()
        f.write(f"{ks} {g} {re:.25f} {im:.25f}\n")
