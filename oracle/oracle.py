"""ctypes front end of the plain FP64 CPU oracle (oracle/fstat_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It never imports the CUDA package
``paper_2407_10797_b200`` and the CUDA package never imports it.

``build()`` compiles the C file with gcc (-O2, no fast-math, OpenMP over particles) into
oracle/libfstat_oracle.so; every function below is a thin marshalling wrapper, the arithmetic is all
in the C file, which cites the PAPER.md passage each step follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fstat_oracle.c")
_LIB = os.path.join(_HERE, "libfstat_oracle.so")
_lock = threading.Lock()
_lib = None


class Options(C.Structure):
    _fields_ = [("f_ref_e0", C.c_double), ("arm_length_m", C.c_double),
                ("orbit_kappa", C.c_double), ("orbit_lambda", C.c_double), ("tdi_channel", C.c_int32)]


TDI_CHANNELS = {"X": 0, "Y": 1, "Z": 2, "A": 3, "E": 4, "T": 5}


def build(force: bool = False) -> str:
    """Compile the oracle if the shared object is missing or older than the source."""
    with _lock:
        if (not force and os.path.exists(_LIB)
                and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
            return _LIB
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
        return _LIB


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.oracle_default_options.argtypes = [C.POINTER(Options)]
        L.oracle_params_valid.argtypes = [C.POINTER(C.c_double)]
        L.oracle_params_valid.restype = C.c_int
        L.oracle_pn_alpha.argtypes = [C.c_double, C.c_double, C.POINTER(C.c_double)]
        L.oracle_phase.argtypes = [C.POINTER(C.c_double), C.c_double, C.POINTER(Options),
                                   C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.oracle_orbit.argtypes = [C.c_double, C.POINTER(Options), C.POINTER(C.c_double)]
        L.oracle_sky_basis.argtypes = [C.c_double, C.c_double] + [C.POINTER(C.c_double)] * 3
        L.oracle_response.argtypes = [C.POINTER(C.c_double), C.c_double, C.c_double, C.POINTER(Options),
                                      C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.oracle_template.argtypes = [C.POINTER(C.c_double), C.c_int64, C.POINTER(C.c_double),
                                      C.POINTER(Options), C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.oracle_inner_products.argtypes = [C.POINTER(C.c_double)] * 4 + [C.c_double, C.c_int64, C.c_int64,
                                            C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.oracle_fstat_from_NM.argtypes = [C.POINTER(C.c_double)] * 4
        L.oracle_fstat_from_NM.restype = C.c_int
        L.oracle_fstat_batch.argtypes = [C.c_int64, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                         C.POINTER(C.c_double), C.c_int32, C.POINTER(C.c_int64), C.c_int64,
                                         C.POINTER(C.c_double), C.POINTER(Options), C.c_int, C.c_int,
                                         C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                         C.POINTER(C.c_int32)]
        L.oracle_fstat_batch.restype = C.c_int
        L.oracle_max_threads.restype = C.c_int
        L.oracle_fstat_partition.argtypes = [C.POINTER(C.c_double)] * 4 + [C.c_double, C.c_int64, C.c_int64, C.c_int,
                                             C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                             C.POINTER(C.c_double)]
        L.oracle_fstat_partition.restype = C.c_int
        L.oracle_fstat_batch_multi.argtypes = [C.c_int64, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                               C.POINTER(C.c_double), C.c_int32, C.POINTER(C.c_int32),
                                               C.POINTER(C.c_int64), C.c_int64, C.POINTER(C.c_double),
                                               C.POINTER(Options), C.c_int, C.c_int, C.POINTER(C.c_double),
                                               C.POINTER(C.c_double)]
        L.oracle_fstat_batch_multi.restype = C.c_int
        L.oracle_template_band.argtypes = [C.POINTER(C.c_double), C.c_int64, C.POINTER(C.c_double), C.c_double,
                                           C.POINTER(Options), C.POINTER(C.c_int64), C.POINTER(C.c_int64),
                                           C.POINTER(C.c_int)]
        _lib = L
    return _lib


def default_options(**kw) -> Options:
    o = Options()
    lib().oracle_default_options(C.byref(o))
    for k, v in kw.items():
        setattr(o, k, v)
    return o


def _opt(o: Optional[Options]) -> Options:
    return default_options() if o is None else o


def _par(p) -> np.ndarray:
    p = np.ascontiguousarray(p, dtype=np.float64)
    assert p.shape[-1] == 6
    return p


def params_valid(par) -> bool:
    return bool(lib().oracle_params_valid(_dp(_par(par))))


def pn_alpha(eta: float, v: float) -> np.ndarray:
    a = np.zeros(7)
    lib().oracle_pn_alpha(float(eta), float(v), _dp(a))
    return a


def phase(par, f: float, opt: Optional[Options] = None) -> Tuple[float, float]:
    """(Psi_0(f), t_f) for one particle at one frequency."""
    psi, tf = C.c_double(), C.c_double()
    lib().oracle_phase(_dp(_par(par)), float(f), C.byref(_opt(opt)), C.byref(psi), C.byref(tf))
    return psi.value, tf.value


def orbit(t: float, opt: Optional[Options] = None) -> np.ndarray:
    """[3][3] spacecraft positions (rows: spacecraft 1, 2, 3) at time t, metres."""
    p = np.zeros((3, 3))
    lib().oracle_orbit(float(t), C.byref(_opt(opt)), _dp(p))
    return p


def sky_basis(theta: float, phi: float):
    k, u, v = np.zeros(3), np.zeros(3), np.zeros(3)
    lib().oracle_sky_basis(float(theta), float(phi), _dp(k), _dp(u), _dp(v))
    return k, u, v


def response(par, f: float, t: float, opt: Optional[Options] = None) -> Tuple[complex, complex]:
    """(T_plus, T_cross) of TDI X at frequency f with the constellation at time t."""
    tp, tc = np.zeros(2), np.zeros(2)
    lib().oracle_response(_dp(_par(par)), float(f), float(t), C.byref(_opt(opt)), _dp(tp), _dp(tc))
    return complex(tp[0], tp[1]), complex(tc[0], tc[1])


def template(par, freq, opt: Optional[Options] = None) -> Tuple[np.ndarray, np.ndarray]:
    """(u_plus, u_cross) complex128 arrays over ``freq`` for one particle."""
    freq = np.ascontiguousarray(freq, dtype=np.float64)
    n = freq.shape[0]
    up, uc = np.zeros(n, dtype=np.complex128), np.zeros(n, dtype=np.complex128)
    lib().oracle_template(_dp(_par(par)), n, _dp(freq), C.byref(_opt(opt)),
                          up.ctypes.data_as(C.POINTER(C.c_double)), uc.ctypes.data_as(C.POINTER(C.c_double)))
    return up, uc


def inner_products(dw, inv_sn, u_plus, u_cross, df: float, lo: int, hi: int, use_ld: bool = False):
    """(N[4], M[4][4]) over bins [lo, hi)."""
    dw = np.ascontiguousarray(dw, dtype=np.complex128)
    inv_sn = np.ascontiguousarray(inv_sn, dtype=np.float64)
    u_plus = np.ascontiguousarray(u_plus, dtype=np.complex128)
    u_cross = np.ascontiguousarray(u_cross, dtype=np.complex128)
    N, M = np.zeros(4), np.zeros((4, 4))
    cd = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    lib().oracle_inner_products(cd(dw), _dp(inv_sn), cd(u_plus), cd(u_cross), float(df), int(lo), int(hi),
                                int(use_ld), _dp(N), _dp(M))
    return N, M


def fstat_from_NM(N, M):
    """(F, a[4], singular_flag) = max_a [a.N - a^T M a / 2]."""
    N = np.ascontiguousarray(N, dtype=np.float64)
    M = np.ascontiguousarray(M, dtype=np.float64)
    F = C.c_double()
    a = np.zeros(4)
    flag = lib().oracle_fstat_from_NM(_dp(N), _dp(M), C.byref(F), _dp(a))
    return F.value, a, int(flag)


def fstat_partition(dw, inv_sn, u_plus, u_cross, df: float, lo: int, hi: int, mode: int = 0):
    """(F, a[4], singular_flag) of one partition [lo, hi) of given templates.  mode 0: compensated double sums,
    1: long-double sums rounded to double, 2: long-double sums handed to the solve unrounded (the reference for
    near-singular M, hazard H3)."""
    dw = np.ascontiguousarray(dw, dtype=np.complex128)
    inv_sn = np.ascontiguousarray(inv_sn, dtype=np.float64)
    u_plus = np.ascontiguousarray(u_plus, dtype=np.complex128)
    u_cross = np.ascontiguousarray(u_cross, dtype=np.complex128)
    cd = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    F = C.c_double()
    a = np.zeros(4)
    flag = lib().oracle_fstat_partition(cd(dw), _dp(inv_sn), cd(u_plus), cd(u_cross), float(df), int(lo), int(hi),
                                        int(mode), C.byref(F), None, None, _dp(a))
    return F.value, a, int(flag)


def fstat_batch(freq, dw, inv_sn, edges, params, opt: Optional[Options] = None, use_ld: bool = False,
                n_threads: int = 0, want_NM: bool = False):
    """F[P], Fk[P][n_part] (and NM[P][n_part][20], flags[P][n_part] when want_NM) for P particles."""
    freq = np.ascontiguousarray(freq, dtype=np.float64)
    dw = np.ascontiguousarray(dw, dtype=np.complex128)
    inv_sn = np.ascontiguousarray(inv_sn, dtype=np.float64)
    edges = np.ascontiguousarray(edges, dtype=np.int64)
    params = _par(params).reshape(-1, 6)
    P, n_part, n = params.shape[0], edges.shape[0] - 1, freq.shape[0]
    assert edges[0] == 0 and edges[-1] == n and np.all(np.diff(edges) > 0)
    F = np.zeros(P)
    Fk = np.zeros((P, n_part))
    NM = np.zeros((P, n_part, 20)) if want_NM else None
    flags = np.zeros((P, n_part), dtype=np.int32)
    rc = lib().oracle_fstat_batch(n, _dp(freq), dw.ctypes.data_as(C.POINTER(C.c_double)), _dp(inv_sn),
                                  n_part, edges.ctypes.data_as(C.POINTER(C.c_int64)), P, _dp(params),
                                  C.byref(_opt(opt)), int(use_ld), int(n_threads), _dp(F), _dp(Fk),
                                  _dp(NM) if want_NM else None, flags.ctypes.data_as(C.POINTER(C.c_int32)))
    if rc != 0:
        raise MemoryError("oracle_fstat_batch: allocation failed")
    if want_NM:
        return F, Fk, NM, flags
    return F, Fk


def fstat_batch_multi(freq, dw, inv_sn, edge_sets, params, opt: Optional[Options] = None, use_ld: bool = False,
                      n_threads: int = 0):
    """[(F[P], Fk[P][n_part_s]) for every edge set]: ``fstat_batch`` for several partition sets over the same data,
    with each particle's templates written out once (bit-equal to one ``fstat_batch`` call per set)."""
    freq = np.ascontiguousarray(freq, dtype=np.float64)
    dw = np.ascontiguousarray(dw, dtype=np.complex128)
    inv_sn = np.ascontiguousarray(inv_sn, dtype=np.float64)
    params = _par(params).reshape(-1, 6)
    sets = [np.ascontiguousarray(e, dtype=np.int64) for e in edge_sets]
    n = freq.shape[0]
    for e in sets:
        assert e[0] == 0 and e[-1] == n and np.all(np.diff(e) > 0)
    P = params.shape[0]
    n_part = np.array([e.shape[0] - 1 for e in sets], dtype=np.int32)
    edges = np.concatenate(sets)
    F = np.zeros((len(sets), P))
    Fk = np.zeros(P * int(n_part.sum()))
    rc = lib().oracle_fstat_batch_multi(n, _dp(freq), dw.ctypes.data_as(C.POINTER(C.c_double)), _dp(inv_sn),
                                        len(sets), n_part.ctypes.data_as(C.POINTER(C.c_int32)),
                                        edges.ctypes.data_as(C.POINTER(C.c_int64)), P, _dp(params),
                                        C.byref(_opt(opt)), int(use_ld), int(n_threads), _dp(F), _dp(Fk))
    if rc != 0:
        raise MemoryError("oracle_fstat_batch_multi: allocation failed")
    out, off = [], 0
    for s, k in enumerate(n_part):
        out.append((F[s].copy(), Fk[off:off + P * int(k)].reshape(P, int(k)).copy()))
        off += P * int(k)
    return out


def template_band(par, freq, T_obs: float, opt: Optional[Options] = None) -> Tuple[int, int]:
    """Row f2: the bins [k_lo, k_hi) of ``freq`` whose stationary time t_f (Eq. 20 :220) lies in
    the observation [0, T_obs]: k_lo = #{t_f < 0}, k_hi = #{t_f <= T_obs}, counted bin by bin."""
    freq = np.ascontiguousarray(freq, dtype=np.float64)
    lo, hi, mono = C.c_int64(), C.c_int64(), C.c_int()
    lib().oracle_template_band(_dp(_par(par)), freq.shape[0], _dp(freq), float(T_obs), C.byref(_opt(opt)),
                               C.byref(lo), C.byref(hi), C.byref(mono))
    assert mono.value == 1, "t_f is not increasing along the grid: the band is not an interval"
    return int(lo.value), int(hi.value)


def band_edges(k_lo: int, k_hi: int, n_bins: int, n_seg: int, lattice: int = 1) -> np.ndarray:
    """Reading A26: the paper fixes only the number of segments and the outer limits (:122).  Here the outer
    limits are rounded to the nearest multiple of ``lattice`` bins (half up), the band is split into n_seg
    parts of equal length in lattice cells up to the floor, e_j = C (q_lo + floor(j (q_hi - q_lo) / n_seg)),
    and every edge is clipped to the grid.  Plain Python integers."""
    Cc = int(lattice)
    q_lo, q_hi = (int(k_lo) + Cc // 2) // Cc, (int(k_hi) + Cc // 2) // Cc
    return np.array([min(Cc * (q_lo + (j * (q_hi - q_lo)) // int(n_seg)), int(n_bins)) for j in range(int(n_seg) + 1)],
                    dtype=np.int64)


def fstat_bands(freq, dw, inv_sn, params, n_seg: int, lattice: int = 1, opt: Optional[Options] = None,
                use_ld: bool = False, want_amp: bool = False):
    """Row f2: the semi-coherent F-statistic with the paper's own segment limits: for every
    particle the template is windowed to its band [k_lo, k_hi) (t_f in [0, T_obs], T_obs = 1/df) and that
    band is cut into n_seg partitions (``band_edges``); F_k from the same inner products and 4x4 solve as
    ``fstat_batch``; an empty partition contributes F_k = 0.  Returns F[P], Fk[P][n_seg], edges[P][n_seg+1]
    (and, with want_amp, the maximising amplitudes a[P][n_seg][4] of Eq. 10 :96; NaN for invalid particles)."""
    freq = np.ascontiguousarray(freq, dtype=np.float64)
    dw = np.ascontiguousarray(dw, dtype=np.complex128)
    inv_sn = np.ascontiguousarray(inv_sn, dtype=np.float64)
    params = _par(params).reshape(-1, 6)
    n = freq.shape[0]
    df = (freq[-1] - freq[0]) / (n - 1)
    P = params.shape[0]
    F, Fk = np.zeros(P), np.zeros((P, n_seg))
    amp = np.zeros((P, n_seg, 4))
    edges = np.zeros((P, n_seg + 1), dtype=np.int64)
    for p in range(P):
        if not params_valid(params[p]):
            F[p], Fk[p], amp[p] = -np.inf, -np.inf, np.nan
            continue
        k_lo, k_hi = template_band(params[p], freq, 1.0 / df, opt)
        e = band_edges(k_lo, k_hi, n, n_seg, lattice)
        edges[p] = e
        if e[-1] <= e[0]:
            continue
        a, b = int(e[0]), int(e[-1])
        up = np.zeros(n, dtype=np.complex128)
        uc = np.zeros(n, dtype=np.complex128)
        up[a:b], uc[a:b] = template(params[p], freq[a:b], opt)
        for j in range(n_seg):
            if e[j + 1] > e[j]:
                N, M = inner_products(dw, inv_sn, up, uc, df, int(e[j]), int(e[j + 1]), use_ld)
                Fk[p, j], amp[p, j], _ = fstat_from_NM(N, M)
        F[p] = float(np.sum(Fk[p].astype(np.longdouble)))
    if want_amp:
        return F, Fk, edges, amp
    return F, Fk, edges


def fstat_batch_channels(freq, channels, edges, params, use_ld: bool = False):
    """Row f4 (Eq. 3: Lambda = sum over TDI combinations I with mutually independent noise of
    <s^I, h^I>_I - |h^I|_I^2 / 2): the four amplitudes are common to all channels, so N^i = sum_I <d_I, A^i_I>_I and
    M^ij = sum_I <A^i_I, A^j_I>_I (Eq. 8-9 per channel), and F_k = max_a [a.N - a^T M a / 2] as before.
    ``channels`` = [(dw_I, inv_sn_I, options_I), ...]; the options carry the channel's response (Y and Z are X with
    the spacecraft relabelled cyclically, i.e. orbit_lambda + 2 pi/3, + 4 pi/3: beta_n = 2 pi n/3 + lambda, reading A9).
    Returns F[P], Fk[P][n_part]."""
    params = _par(params).reshape(-1, 6)
    edges = np.ascontiguousarray(edges, dtype=np.int64)
    P, n_part = params.shape[0], edges.shape[0] - 1
    NM = None
    for dw, inv_sn, opt in channels:
        _, _, nm, _ = fstat_batch(freq, dw, inv_sn, edges, params, opt, use_ld=use_ld, want_NM=True)
        NM = nm if NM is None else NM + nm
    F, Fk = np.zeros(P), np.zeros((P, n_part))
    for p in range(P):
        if not params_valid(params[p]):
            F[p], Fk[p] = -np.inf, -np.inf
            continue
        for k in range(n_part):
            Fk[p, k] = fstat_from_NM(NM[p, k, :4], NM[p, k, 4:].reshape(4, 4))[0]
        F[p] = float(np.sum(Fk[p].astype(np.longdouble)))
    return F, Fk


def max_threads() -> int:
    return int(lib().oracle_max_threads())
