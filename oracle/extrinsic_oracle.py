"""Plain restatement of PAPER.md App. B (:409-442): Eq. B1 (extrinsic parameters -> the four amplitudes) and Eq. B2-B3
(amplitudes -> D_L, iota, psi, phi_c), as printed.  TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/ may import it; it
shares nothing with paper_2407_10797_b200/ (whose C function fstat_extrinsic_from_amplitudes it checks).

Pins (tests/test_extrinsic.py, CPU): B2-B3 invert B1 on random parameter sets inside the principal branches; outside
them the recovered set reproduces the amplitudes through B1; D_L = 2 / A and iota are branch-free.  P20: amplitudes
estimated from a quadrupole-formula binary's time-domain TDI signal (tests/td_sim.py PhysicalBinary) come back as its
physical distance (5 %) and inclination (0.05 rad).

Reading A25: Eq. B2's plain arctan fixes phi_c only modulo pi, while phi_c -> phi_c + pi flips the sign of
all four a_i in Eq. B1.  `b2_b3` takes the paper's arctan values and adds pi to phi_c when that is what reproduces the
sign of the amplitudes; psi stays in the paper's branch (-pi/4, pi/4].
"""
import math

import numpy as np


def b1(d_l, psi, iota, phi_c):
    """Eq. B1 (:413-420) as printed."""
    p = (1.0 + math.cos(iota) ** 2) / 2.0
    ci = math.cos(iota)
    a1 = (math.cos(2 * psi) * p * math.cos(phi_c) - math.sin(2 * psi) * ci * math.sin(phi_c)) / d_l
    a2 = -(math.sin(2 * psi) * p * math.cos(phi_c) + math.cos(2 * psi) * ci * math.sin(phi_c)) / d_l
    a3 = -(math.cos(2 * psi) * p * math.sin(phi_c) + math.sin(2 * psi) * ci * math.cos(phi_c)) / d_l
    a4 = (math.sin(2 * psi) * p * math.sin(phi_c) - math.cos(2 * psi) * ci * math.cos(phi_c)) / d_l
    return np.array([a1, a2, a3, a4])


def b2_b3(a):
    """Eq. B3 then Eq. B2 (:426-440) as printed, in fp64: returns (D_L, iota, psi, phi_c)."""
    a1, a2, a3, a4 = (float(x) for x in a)
    s1 = math.sqrt((a1 + a4) ** 2 + (a2 - a3) ** 2)
    s2 = math.sqrt((a1 - a4) ** 2 + (a2 + a3) ** 2)
    A_plus = s1 + s2                                                           # Eq. B3
    A_cross = s1 - s2
    A = A_plus + math.sqrt(max(A_plus ** 2 - A_cross ** 2, 0.0))
    d_l = 2.0 / A                                                              # Eq. B2
    iota = math.acos(max(-1.0, min(1.0, -A_cross / (A_plus + math.sqrt(max(A_plus ** 2 - A_cross ** 2, 0.0))))))
    num = A_plus * a4 - A_cross * a1
    den = -(A_cross * a2 + A_plus * a3)
    psi = 0.5 * (math.atan(num / den) if den != 0.0 else math.copysign(math.pi / 2.0, num))
    c = 1.0 if math.sin(2.0 * psi) >= 0.0 else -1.0
    den_c = -c * (A_cross * a3 + A_plus * a2)
    phi_c = math.atan(c * num / den_c) if den_c != 0.0 else math.copysign(math.pi / 2.0, c * num)
    if float(np.dot(b1(d_l, psi, iota, phi_c), [a1, a2, a3, a4])) < 0.0:       # reading A25
        phi_c = phi_c + math.pi if phi_c <= 0.0 else phi_c - math.pi
    return d_l, iota, psi, phi_c
