"""Extrinsic-parameter recovery (App. B): marshalling for the library's host functions
``fstat_extrinsic_from_amplitudes`` (Eq. B2-B3: (D_L, iota, psi, phi_c) from the four maximum-likelihood amplitudes
a = M^-1 N that ``fstat_eval_amplitudes`` returns) and ``fstat_amplitudes_from_extrinsic`` (Eq. B1, the forward map).
No arithmetic of the method here; see include/fstat.h for conventions (readings A21, A25)."""
from __future__ import annotations

import ctypes as C
from typing import Dict, Optional

import numpy as np

from .binding import FstatError, load_library


def extrinsic_from_amplitudes(a, chirp_mass_msun: Optional[float] = None) -> Dict[str, float]:
    """``a`` = (a_1, a_2, a_3, a_4).  With ``chirp_mass_msun`` the amplitudes are the library's (amplitude constant of
    Eq. A2 restored, D_L in metres); without, the paper's a_i (D_L in their inverse units)."""
    v = np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(4))
    out = np.zeros(4)
    st = load_library().fstat_extrinsic_from_amplitudes(v.ctypes.data_as(C.POINTER(C.c_double)),
                                                        float(chirp_mass_msun) if chirp_mass_msun is not None else 0.0,
                                                        out.ctypes.data_as(C.POINTER(C.c_double)))
    if st != 0:
        raise FstatError(st, "fstat_extrinsic_from_amplitudes")
    return {"D_L": float(out[0]), "iota": float(out[1]), "psi": float(out[2]), "phi_c": float(out[3])}


def amplitudes_from_extrinsic(d_l: float, psi: float, iota: float, phi_c: float) -> np.ndarray:
    """Eq. B1 (:413-420) with D_L in the inverse units of the amplitudes."""
    out = np.zeros(4)
    st = load_library().fstat_amplitudes_from_extrinsic(float(d_l), float(psi), float(iota), float(phi_c),
                                                        out.ctypes.data_as(C.POINTER(C.c_double)))
    if st != 0:
        raise FstatError(st, "fstat_amplitudes_from_extrinsic")
    return out
