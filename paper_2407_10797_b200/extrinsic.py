"""Extrinsic-parameter recovery (App. B, Eq. B2-B3): (D_L, iota, psi, phi_c) from the four
maximum-likelihood amplitudes a = M^-1 N that ``fstat_eval_amplitudes`` returns.  Host-side, a few lines of
arithmetic on ONE amplitude vector (the best particle of the final coherent stage): not on the hot path.

The library's templates drop the amplitude constant of Eq. A2 (:402; reading A21),
A = -sqrt(5/24) M_c^(5/6) / (pi^(2/3) D_L), so its amplitudes are K_A times the paper's a_i with
K_A = -sqrt(5/24) (G M_c / c^3)^(5/6) / pi^(2/3) and D_L in seconds; ``chirp_mass_msun`` restores it.
"""
from __future__ import annotations

import math
from typing import Dict, Optional

import numpy as np

GMSUN_C3 = 4.925490947641267e-6      # G Msun / c^3 [s]
C_LIGHT = 299792458.0                # m / s


def amplitude_constant(chirp_mass_msun: float) -> float:
    """K_A of the module docstring [s^(5/6)]: library amplitude = K_A x (paper's a_i with D_L in seconds)."""
    return -math.sqrt(5.0 / 24.0) * (chirp_mass_msun * GMSUN_C3) ** (5.0 / 6.0) / math.pi ** (2.0 / 3.0)


def extrinsic_from_amplitudes(a, chirp_mass_msun: Optional[float] = None) -> Dict[str, float]:
    """Eq. B2-B3 (:426-440).  ``a`` = (a_1, a_2, a_3, a_4).  Returns iota, psi in (-pi/4, pi/4] (the branch of
    the paper's arctan), phi_c in (-pi, pi] (the paper's arctan plus the half-plane that reproduces the sign of
    the amplitudes) and D_L: in metres when ``chirp_mass_msun`` is given,
    else 2 / A in the inverse units of ``a``."""
    a1, a2, a3, a4 = (float(x) for x in np.asarray(a, dtype=np.float64).reshape(4))
    if chirp_mass_msun is not None:
        k = amplitude_constant(chirp_mass_msun)
        a1, a2, a3, a4 = a1 / k, a2 / k, a3 / k, a4 / k
    r_plus = math.hypot(a1 + a4, a2 - a3)
    r_minus = math.hypot(a1 - a4, a2 + a3)
    A_plus = r_plus + r_minus
    A_cross = r_plus - r_minus
    root = 2.0 * math.sqrt(r_plus * r_minus)          # = sqrt(A_+^2 - A_x^2) of Eq. B3, without the cancellation
    A = A_plus + root
    iota = math.acos(max(-1.0, min(1.0, -A_cross / A))) if A > 0.0 else 0.0
    num = A_plus * a4 - A_cross * a1
    den_psi = -(A_cross * a2 + A_plus * a3)
    psi = 0.5 * (math.atan(num / den_psi) if den_psi != 0.0 else math.copysign(math.pi / 2.0, num))
    c = 1.0 if math.sin(2.0 * psi) >= 0.0 else -1.0
    den = -c * (A_cross * a3 + A_plus * a2)
    phi_c = math.atan(c * num / den) if den != 0.0 else math.copysign(math.pi / 2.0, c * num)
    # Eq. B2's arctan fixes phi_c only modulo pi, and phi_c -> phi_c + pi flips the sign of all four a_i in
    # Eq. B1: the half-plane is the one that reproduces the sign of the amplitudes (reading A25).
    if A > 0.0 and float(np.dot(amplitudes_from_extrinsic(2.0 / A, psi, iota, phi_c), [a1, a2, a3, a4])) < 0.0:
        phi_c = phi_c + math.pi if phi_c <= 0.0 else phi_c - math.pi
    d_l = 2.0 / A if A > 0.0 else math.inf
    if chirp_mass_msun is not None:
        d_l *= C_LIGHT
    return {"D_L": d_l, "iota": iota, "psi": psi, "phi_c": phi_c}


def amplitudes_from_extrinsic(d_l: float, psi: float, iota: float, phi_c: float) -> np.ndarray:
    """Eq. B1 (:413-420), the forward map, with D_L in the inverse units of the amplitudes."""
    p = 0.5 * (1.0 + math.cos(iota) ** 2)
    ci = math.cos(iota)
    c2, s2 = math.cos(2.0 * psi), math.sin(2.0 * psi)
    cp, sp = math.cos(phi_c), math.sin(phi_c)
    return np.array([(c2 * p * cp - s2 * ci * sp), -(s2 * p * cp + c2 * ci * sp),
                     -(c2 * p * sp + s2 * ci * cp), (s2 * p * sp - c2 * ci * cp)]) / d_l
