"""Pins P15-P17: the 2.5PN / 3PN coefficients alpha_5, alpha_6 and the eccentric constant 2355/1462 of the
oracle's Psi_0 (PAPER.md:404 Eq. A3; the paper prints none of them: "details in [85-88]", :407) against
INDEPENDENT statements of the literature the paper cites -- none of them retypes Eq. A3's coefficients:

  P15  t_f = (1/2pi) dPsi_0/df (Eq. 20 :220) against the 3PN TaylorT2 time series t(v) of ref. [88]
       (Buonanno, Iyer, Ochsner, Pan, Sathyaprakash 2009, :543; its Eq. 3.8b), typed here from that paper.
       The stationary-phase relation makes the two agree TERM BY TERM (both are the same truncated E'(v)/F(v)
       integrated once or twice), so the tolerance is rounding, not "next PN order".
  P16  Psi_0 itself against 2 pi f t(v) - 2 phi_orb(v) - pi/4 with TaylorT2's t(v) and orbital phase phi(v)
       (Eq. 3.8a of the same reference).  This also fixes what t_f cannot see: the constant part of alpha_5
       (the "1 +" and v_lso = 6^(-1/2)).
  P17  the eccentric term against Peters' (1964) exact time to coalescence of an eccentric binary,
       T(a_0, e_0) = (12/19) (c_0^4 / beta) int_0^e0 e^(29/19) [1 + (121/304) e^2]^(1181/2299) (1 - e^2)^(-3/2) de,
       by numerical quadrature: to O(e^2) it is T_circ [1 - (157/43) e^2], and the oracle's
       -(3/128)(pi Mc f)^(-5/3) (2355/1462) e0^2 (f_ref/f)^(19/9) gives, through the derivative,
       3 * 34 * 2355 / (5 * 9 * 1462) = 157/43; the exponent 19/9 is Peters' e ~ f^(-19/18).

`test_corrupted_coefficients_fail_the_pins` is the proof that the pins bite: scratch copies of
oracle/fstat_oracle.c with one constant corrupted each (alpha_5's rational, its log argument, alpha_6's
rational / eta sign / log argument / Euler term, 2355/1462, the exponent 19/9) are compiled into a temporary
directory and every one of them must fail at least one of P15-P17.  CPU only.
"""
import ctypes as C
import math
import os
import re
import subprocess

import numpy as np
import pytest
from scipy import integrate

GMSUN = 4.925490947641267e-6
EULER = 0.5772156649015329
HERE = os.path.dirname(os.path.abspath(__file__))
ORACLE_C = os.path.join(os.path.dirname(HERE), "oracle", "fstat_oracle.c")


# ------------------------------------------------------------------ TaylorT2 of ref. [88], Eq. 3.8a / 3.8b
def taylor_t2_time(v, eta, M):
    """t_ref - t(v) [s]: time to coalescence at PN velocity v, 3PN, non-spinning (ref. [88] Eq. 3.8b)."""
    pi = math.pi
    s = (1.0
         + (743.0 / 252.0 + 11.0 / 3.0 * eta) * v ** 2
         - 32.0 / 5.0 * pi * v ** 3
         + (3058673.0 / 508032.0 + 5429.0 / 504.0 * eta + 617.0 / 72.0 * eta ** 2) * v ** 4
         - (7729.0 / 252.0 - 13.0 / 3.0 * eta) * pi * v ** 5
         + (-10052469856691.0 / 23471078400.0 + 128.0 / 3.0 * pi ** 2 + 6848.0 / 105.0 * EULER
            + (3147553127.0 / 3048192.0 - 451.0 / 12.0 * pi ** 2) * eta
            - 15211.0 / 1728.0 * eta ** 2 + 25565.0 / 1296.0 * eta ** 3
            + 3424.0 / 105.0 * math.log(16.0 * v ** 2)) * v ** 6)
    return 5.0 * M / (256.0 * eta * v ** 8) * s


def taylor_t2_orbital_phase(v, eta):
    """phi_ref - phi(v) [rad]: ORBITAL phase to coalescence, 3PN (ref. [88] Eq. 3.8a); GW phase = twice this."""
    pi = math.pi
    v_lso = 1.0 / math.sqrt(6.0)
    s = (1.0
         + (3715.0 / 1008.0 + 55.0 / 12.0 * eta) * v ** 2
         - 10.0 * pi * v ** 3
         + (15293365.0 / 1016064.0 + 27145.0 / 1008.0 * eta + 3085.0 / 144.0 * eta ** 2) * v ** 4
         + (38645.0 / 672.0 - 65.0 / 8.0 * eta) * math.log(v / v_lso) * pi * v ** 5
         + (12348611926451.0 / 18776862720.0 - 160.0 / 3.0 * pi ** 2 - 1712.0 / 21.0 * EULER
            + (-15737765635.0 / 12192768.0 + 2255.0 / 48.0 * pi ** 2) * eta
            + 76055.0 / 6912.0 * eta ** 2 - 127825.0 / 5184.0 * eta ** 3
            - 856.0 / 21.0 * math.log(16.0 * v ** 2)) * v ** 6)
    return s / (32.0 * eta * v ** 5)


# (M_c [Msun], eta, f [Hz]) spanning v = 0.016 .. 0.33: the paper's range (M_c 20-80, 10-50 mHz, v < 0.05) and a
# strong-field stretch where the 2.5PN / 3PN terms are percent-level pieces of the series
CASES = [(20.0, 0.25, 0.01), (30.0, 0.24, 0.02), (80.0, 0.2, 0.05), (40.0, 0.1, 0.1),
         (3.0e4, 0.25, 0.01), (3.0e4, 0.16, 0.02), (1.0e5, 0.21, 0.015), (3.0e5, 0.25, 0.008)]


def _v_of(Mc, eta, f):
    M = Mc * GMSUN * eta ** -0.6
    return (math.pi * M * f) ** (1.0 / 3.0), M


def check_p15(phase):
    """phase(par, f) -> (Psi_0, t_f).  Raises AssertionError when t_f is not TaylorT2's t(v)."""
    vs = []
    for Mc, eta, f in CASES:
        v, M = _v_of(Mc, eta, f)
        vs.append(v)
        par = np.array([0.0, Mc, eta, 1.0, 2.0, 0.0])
        tau_orc = -phase(par, f)[1]                        # t_c = 0: t_f = -tau
        tau_t2 = taylor_t2_time(v, eta, M)
        # the two series are the same polynomial in v: rounding only.  The 3PN term is 1e-8 (v = 0.016) to
        # 5e-3 (v = 0.3) of tau and the 2.5PN term 3e-7 .. 0.2: a wrong alpha_5 or alpha_6 cannot hide below 1e-11
        assert tau_orc == pytest.approx(tau_t2, rel=1e-11), (Mc, eta, f, v)
    assert min(vs) < 0.02 and max(vs) > 0.25


def check_p16(phase):
    """Psi_0 = 2 pi f t(f) - 2 phi_orb(f) - pi/4 with t_c = 0, phi_c = 0 (stationary phase, A5 convention)."""
    for Mc, eta, f in CASES:
        v, M = _v_of(Mc, eta, f)
        par = np.array([0.0, Mc, eta, 1.0, 2.0, 0.0])
        psi_orc = phase(par, f)[0]
        psi_t2 = 2.0 * math.pi * f * (-taylor_t2_time(v, eta, M)) + 2.0 * taylor_t2_orbital_phase(v, eta) - math.pi / 4.0
        scale = abs(2.0 * taylor_t2_orbital_phase(v, eta)) + abs(2.0 * math.pi * f * taylor_t2_time(v, eta, M))   # rounding scale of the two pieces
        assert abs(psi_orc - psi_t2) < 2e-13 * scale + 1e-12, (Mc, eta, f, v, psi_orc - psi_t2)


def peters_time_ratio(e0):
    """T(a_0, e_0) / T_circ(a_0) from Peters 1964 Eq. 5.11 / 5.14 by quadrature (a_0 = the same semi-major axis)."""
    g = lambda e: e ** (29.0 / 19.0) * (1.0 + 121.0 / 304.0 * e * e) ** (1181.0 / 2299.0) / (1.0 - e * e) ** 1.5
    integral = integrate.quad(g, 0.0, e0, epsabs=0.0, epsrel=1e-13)[0]
    # a(e) = c_0 e^(12/19) (1 + 121/304 e^2)^(870/2299) / (1 - e^2);  T_circ = a_0^4 / (4 beta)
    a0_over_c0 = e0 ** (12.0 / 19.0) * (1.0 + 121.0 / 304.0 * e0 * e0) ** (870.0 / 2299.0) / (1.0 - e0 * e0)
    return (12.0 / 19.0) * integral / (a0_over_c0 ** 4 / 4.0)


def check_p17(phase_with_fref):
    """phase_with_fref(par, f, f_ref) -> (Psi_0, t_f).  The eccentric shift of the time to coalescence at
    frequency f, for an orbit of eccentricity e_f there, is Peters' T/T_circ - 1 = -(157/43) e_f^2 + O(e_f^4);
    e_f = e0 (f_ref/f)^(19/18) by Peters' a(e) at small e (a ~ e^(12/19), f ~ a^(-3/2))."""
    Mc, eta, tc = 30.0, 0.24, 1.1e8
    tau_newt = lambda f: 5.0 / 256.0 * (Mc * GMSUN) ** (-5.0 / 3.0) * (math.pi * f) ** (-8.0 / 3.0)
    for f_ref, f, e0 in ((0.01, 0.01, 0.01), (0.01, 0.01, 0.02), (0.01, 0.03, 0.05), (0.02, 0.012, 0.01), (0.01, 0.004, 0.004)):
        p0 = np.array([tc, Mc, eta, 1.0, 2.0, 0.0])
        p1 = p0.copy(); p1[5] = e0
        shift = (tc - phase_with_fref(p1, f, f_ref)[1]) - (tc - phase_with_fref(p0, f, f_ref)[1])   # tau(e0) - tau(0)
        e_f = e0 * (f_ref / f) ** (19.0 / 18.0)
        want = peters_time_ratio(e_f) - 1.0
        assert want == pytest.approx(-157.0 / 43.0 * e_f ** 2, rel=20.0 * e_f ** 2)          # Peters' own small-e limit
        assert shift / tau_newt(f) == pytest.approx(want, rel=30.0 * e_f ** 2 + 1e-7), (f_ref, f, e0)


# ------------------------------------------------------------------ the oracle as it stands
def _phase_fref(orc):
    return lambda par, f, f_ref: orc.phase(par, f, orc.default_options(f_ref_e0=f_ref))


def test_p15_time_to_coalescence_is_taylor_t2_to_3pn(orc):
    check_p15(orc.phase)


def test_p16_phase_is_the_stationary_phase_transform_of_taylor_t2(orc):
    check_p16(orc.phase)


def test_p17_eccentric_term_is_peters_time_to_coalescence(orc):
    check_p17(_phase_fref(orc))


def test_taylor_t2_series_typed_here_are_mutually_consistent():
    """Guards the pins themselves: the two TaylorT2 series typed above are integrals of the same truncated
    E'(v)/F(v), so d phi_orb / dv = (v^3 / M) dt / dv holds term by term (phi_k = (5/8) (k-8)/(k-5) tau_k); checked by
    central differences up to v = 0.4, where a mistyped digit in any coefficient of either series is >= 1e-4."""
    M = 1.0
    for eta in (0.1, 0.22, 0.25):
        for v in (0.05, 0.1, 0.2, 0.4):
            h = 1e-4 * v
            dphi = (taylor_t2_orbital_phase(v - h, eta) - taylor_t2_orbital_phase(v + h, eta)) / (2 * h)   # d phi / dv
            dt = (taylor_t2_time(v - h, eta, M) - taylor_t2_time(v + h, eta, M)) / (2 * h)                 # d t / dv
            assert abs(dphi / dt / (v ** 3 / M) - 1.0) < 1e-6, (eta, v)


# ------------------------------------------------------------------ the pins bite: corrupted scratch copies
class _Opt(C.Structure):
    _fields_ = [("f_ref_e0", C.c_double), ("arm_length_m", C.c_double), ("orbit_kappa", C.c_double),
                ("orbit_lambda", C.c_double), ("tdi_channel", C.c_int32)]


def _compile_phase(src_text, workdir, tag):
    c_path = os.path.join(workdir, "orc_%s.c" % tag)
    so_path = os.path.join(workdir, "orc_%s.so" % tag)
    with open(c_path, "w") as fh:
        fh.write(src_text)
    subprocess.run(["gcc", "-O1", "-std=c11", "-ffp-contract=off", "-shared", "-fPIC", "-o", so_path, c_path, "-lm"],
                   check=True)
    lib = C.CDLL(so_path)
    lib.oracle_phase.argtypes = [C.POINTER(C.c_double), C.c_double, C.POINTER(_Opt), C.POINTER(C.c_double),
                                 C.POINTER(C.c_double)]

    def phase(par, f, f_ref=0.01):
        par = np.ascontiguousarray(par, dtype=np.float64)
        o = _Opt(f_ref, 2.5e9, 0.0, 0.0, 0)
        psi, tf = C.c_double(), C.c_double()
        lib.oracle_phase(par.ctypes.data_as(C.POINTER(C.c_double)), float(f), C.byref(o), C.byref(psi), C.byref(tf))
        return psi.value, tf.value
    return phase


MUTATIONS = [
    ("alpha5_rational", "38645.0 / 756.0", "38645.0 / 765.0"),
    ("alpha5_eta", "65.0 * eta / 9.0", "56.0 * eta / 9.0"),
    ("alpha5_log_argument", "log(v / v_lso)", "log(v * v_lso)"),
    ("alpha5_constant_part", "(1.0 + 3.0 * log(v / v_lso))", "(3.0 * log(v / v_lso))"),
    ("alpha6_rational", "11583231236531.0 / 4694215680.0", "11583231236351.0 / 4694215680.0"),
    ("alpha6_pi2", "640.0 * pi * pi / 3.0", "640.0 * pi * pi / 9.0"),
    ("alpha6_euler", "6848.0 * ORC_EULER / 21.0", "6848.0 * ORC_EULER / 12.0"),
    ("alpha6_eta_sign", "+ eta * (-15737765635.0 / 3048192.0", "- eta * (-15737765635.0 / 3048192.0"),
    ("alpha6_eta_pi2", "2255.0 * pi * pi / 12.0", "2255.0 * pi * pi / 21.0"),
    ("alpha6_eta3", "127825.0 * eta * eta * eta / 1296.0", "127825.0 * eta * eta * eta / 1269.0"),
    ("alpha6_log_argument", "log(4.0 * v)", "log(2.0 * v)"),
    ("alpha6_log_coefficient", "6848.0 / 21.0", "6848.0 / 12.0"),
    ("eccentric_constant", "2355.0 / 1462.0", "2355.0 / 1426.0"),
    ("eccentric_exponent", "19.0 / 9.0", "19.0 / 6.0"),
]


def _fails(check, *args):
    try:
        check(*args)
    except AssertionError:
        return True
    return False


def test_corrupted_coefficients_fail_the_pins(tmp_path):
    src = open(ORACLE_C).read()
    src = re.sub(r"#pragma omp[^\n]*\n", "\n", src)            # the scratch copies need no OpenMP
    good = _compile_phase(src, str(tmp_path), "good")
    fr = lambda ph: (lambda par, f, f_ref: ph(par, f, f_ref))
    check_p15(good); check_p16(good); check_p17(fr(good))      # the unmodified copy passes all three
    for tag, old, new in MUTATIONS:
        assert old in src, tag
        bad_src = src.replace(old, new)
        if tag == "eccentric_exponent":                         # keep the derivative consistent with the phase:
            bad_src = bad_src.replace("(34.0 / 9.0) * pow(f, -43.0 / 9.0)", "(29.0 / 6.0) * pow(f, -35.0 / 6.0)")   # 5/3 + 19/6
        bad = _compile_phase(bad_src, str(tmp_path), tag)
        caught = [name for name, chk, arg in (("P15", check_p15, bad), ("P16", check_p16, bad), ("P17", check_p17, fr(bad)))
                  if _fails(chk, arg)]
        assert caught, "corruption %r passes P15-P17" % tag
        constant_phase = tag in ("alpha5_constant_part", "alpha5_log_argument")   # v_lso only moves a constant phase
        if tag.startswith("alpha") and not constant_phase:
            assert "P15" in caught and "P16" in caught, (tag, caught)
        if constant_phase:
            assert caught == ["P16"], (tag, caught)             # invisible to t_f (and to F: absorbed by phi_c)
        if tag.startswith("eccentric"):
            assert caught == ["P17"], (tag, caught)
