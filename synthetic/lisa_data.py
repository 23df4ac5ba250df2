"""Seeded synthetic LISA TDI-X data sets shaped like the paper's.

The paper analyses 2.5 yr of one simulated TDI-X series (its own noise realisations are not
available); BASELINE.json fixes five synthetic configs that stand in for it.  This module
builds exactly those: grid, analytic PSD, seeded noise, partition edges, particle draws.
It contains no waveform / response / F-statistic arithmetic -- the injection template is
passed in by the caller (``template_fn``), see ``synthetic/__init__.py``.

Recipe (stated again in DESIGN.md, "Synthetic inputs"):
  grid      f_k = k/T, k in [ceil(f_lo T), floor(f_hi T))
  PSD       S_X(f) = 16 sin^2(2 pi f L/c) [S_oms + (3 + cos(4 pi f L/c)) S_acc]
            S_oms = (15e-12 * 2 pi f / c)^2 [1 + (2 mHz/f)^4]
            S_acc = (3e-15 / (2 pi f c))^2 [1 + (0.4 mHz/f)^2][1 + (f/8 mHz)^4]   (reading A8)
  noise     n_k = sqrt(S_X(f_k) T / 4) (x_k + i y_k),  (x, y) = default_rng(seed).standard_normal((N, 2))
            (reading A17: then <n, h> has variance <h, h> for the rectangle-rule inner product)
  particles default_rng(100 + config index); columns drawn in the order tc, Mc, eta, cos(theta), phi, e0
"""
from __future__ import annotations

import dataclasses
import math
from typing import Callable, Optional, Sequence, Tuple

import numpy as np

YEAR_S = 31557600.0          # Julian year (reading A23)
C_SI = 299792458.0
ARM_LENGTH_M = 2.5e9

# config-0 search ranges (BASELINE.json configs[0]); tc range is [T, T + 5 yr]
MC_RANGE = (20.0, 40.0)
ETA_RANGE = (0.2, 0.25)
E0_RANGE = (0.0, 0.1)
TC_SPAN_YR = 5.0

# injection (BASELINE.json configs[1]; angles and extrinsics from PAPER.md:251-260 Table I)
_INJ = dict(Mc=30.0, eta=0.24, e0=0.05, theta=0.7854, phi=2.1216,
            iota=0.5329, psi=1.2501, phic=0.8419, snr=12.0)


@dataclasses.dataclass(frozen=True)
class Config:
    index: int
    name: str
    T: float                      # observation time [s]
    f_lo: float
    f_hi: float
    n_part: Tuple[int, ...]       # N_p values this config is evaluated with
    P: Tuple[int, ...]            # particle counts (one entry except for the wide-band sweep)
    tc_inj: float                 # injected coalescence time [s from data start]
    particle_rule: str            # "wide" | "swarms" | "final"
    noise_seed: int = 0

    @property
    def particle_seed(self) -> int:
        return 100 + self.index


_T_TINY = float(2 ** 20)
_T_25 = 2.5 * YEAR_S             # 78 894 000 s

CONFIGS: Tuple[Config, ...] = (
    Config(0, "tiny", _T_TINY, 0.010, 0.012, (4,), (64,), _T_TINY + YEAR_S, "wide"),
    Config(1, "first_stage", _T_25, 0.01, 0.03, (1024,), (2048,), 3.5 * YEAR_S, "wide"),
    Config(2, "middle_stages", _T_25, 0.01, 0.03, (256, 64, 16), (8192,), 3.5 * YEAR_S, "swarms"),
    Config(3, "final_coherent", _T_25, 0.01, 0.03, (1,), (4096,), 3.5 * YEAR_S, "final"),
    Config(4, "wide_band", _T_25, 0.01, 0.1, (1, 16, 1024), (256, 1024, 4096, 16384, 65536),
           3.5 * YEAR_S, "wide"),
)


# Row f2 (the paper's own segment limits) needs templates whose band [f(t=0), f(t=T)] falls
# inside the grid; the tiny config has none (its particles reach 12.66 mHz at the lowest).  A half-year
# grid small enough for the oracle, with particles whose bands start below, inside and above the grid
# and some that merge during the observation.  Not one of BASELINE.json's five configs.
_T_BANDS = float(2 ** 24)
BANDS_SMALL = Config(5, "bands_small", _T_BANDS, 0.020, 0.026, (1, 4, 16), (64,), 2.0 * YEAR_S, "bands")


def config_by_name(name) -> Config:
    for c in CONFIGS + (BANDS_SMALL,):
        if c.name == name or str(c.index) == str(name):
            return c
    raise KeyError(name)


def frequency_grid(T: float, f_lo: float, f_hi: float) -> Tuple[int, int, np.ndarray]:
    """k_lo, n_bins and f_k = k/T for k in [ceil(f_lo T), floor(f_hi T))."""
    k_lo = int(math.ceil(round(f_lo * T, 6)))
    k_hi = int(math.floor(round(f_hi * T, 6)))
    k = np.arange(k_lo, k_hi, dtype=np.float64)
    return k_lo, k_hi - k_lo, k / T


def psd_tdi_x(f: np.ndarray, L: float = ARM_LENGTH_M) -> np.ndarray:
    """One-sided PSD of first-generation TDI X in fractional-frequency units (reading A8)."""
    f = np.asarray(f, dtype=np.float64)
    x = 2.0 * np.pi * f * L / C_SI
    s_oms = (15e-12 * 2.0 * np.pi * f / C_SI) ** 2 * (1.0 + (2e-3 / f) ** 4)
    s_acc = (3e-15 / (2.0 * np.pi * f * C_SI)) ** 2 * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8e-3) ** 4)
    return 16.0 * np.sin(x) ** 2 * (s_oms + (3.0 + np.cos(2.0 * x)) * s_acc)


def psd_tdi(f: np.ndarray, channel: str = "X", L: float = ARM_LENGTH_M) -> np.ndarray:
    """One-sided PSD of the first-generation TDI combination ``channel`` for equal arms and the noise levels of
    reading A8.  X, Y, Z: ``psd_tdi_x``.  With the cross-spectrum S_XY = -8 sin^2 x cos x [S_oms + 4 S_acc] of two
    Michelson combinations, A = (Z - X)/sqrt 2 and E = (X - 2Y + Z)/sqrt 6 have S_X - S_XY and T = (X + Y + Z)/sqrt 3
    has S_X + 2 S_XY (the combinations with mutually independent noise of PAPER.md:48):
        S_A = S_E = 8 sin^2 x [(2 + cos x) S_oms + 2 (3 + 2 cos x + cos 2x) S_acc],
        S_T = 16 sin^2 x (1 - cos x) S_oms + 128 sin^2 x sin^4(x/2) S_acc,      x = 2 pi f L / c."""
    if channel in ("X", "Y", "Z"):
        return psd_tdi_x(f, L)
    f = np.asarray(f, dtype=np.float64)
    x = 2.0 * np.pi * f * L / C_SI
    s_oms = (15e-12 * 2.0 * np.pi * f / C_SI) ** 2 * (1.0 + (2e-3 / f) ** 4)
    s_acc = (3e-15 / (2.0 * np.pi * f * C_SI)) ** 2 * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8e-3) ** 4)
    if channel in ("A", "E"):
        return 8.0 * np.sin(x) ** 2 * ((2.0 + np.cos(x)) * s_oms + 2.0 * (3.0 + 2.0 * np.cos(x) + np.cos(2.0 * x)) * s_acc)
    if channel == "T":
        return 16.0 * np.sin(x) ** 2 * (1.0 - np.cos(x)) * s_oms + 128.0 * np.sin(x) ** 2 * np.sin(0.5 * x) ** 4 * s_acc
    raise ValueError(channel)


def coloured_noise(sn: np.ndarray, T: float, seed: int) -> np.ndarray:
    """n_k = sqrt(S_n T / 4) (x + i y), (x, y) standard normal (reading A17)."""
    xy = np.random.default_rng(seed).standard_normal((sn.shape[0], 2))
    return np.sqrt(sn * T / 4.0) * (xy[:, 0] + 1j * xy[:, 1])


def equal_bin_edges(n_bins: int, n_part: int) -> np.ndarray:
    """e_j = floor(j n_bins / n_part), j = 0..n_part ("equal-bin partitions", BASELINE.json)."""
    j = np.arange(n_part + 1, dtype=np.int64)
    return (j * np.int64(n_bins)) // np.int64(n_part)


def injection_params(cfg: Config) -> np.ndarray:
    """Intrinsic parameters of the injection in the API order (tc, Mc, eta, theta, phi, e0)."""
    return np.array([cfg.tc_inj, _INJ["Mc"], _INJ["eta"], _INJ["theta"], _INJ["phi"], _INJ["e0"]])


def injection_amplitudes() -> np.ndarray:
    """a_1..a_4 of PAPER.md:413-420 (Eq. B1) for the injected iota, psi, phi_c with D_L = 1.

    Only their ratios matter: the data set rescales the injection to the requested SNR.
    """
    ci = math.cos(_INJ["iota"])
    ap = 0.5 * (1.0 + ci * ci)
    c2, s2 = math.cos(2 * _INJ["psi"]), math.sin(2 * _INJ["psi"])
    cc, sc = math.cos(_INJ["phic"]), math.sin(_INJ["phic"])
    return np.array([c2 * ap * cc - s2 * ci * sc,
                     -(s2 * ap * cc + c2 * ci * sc),
                     -(c2 * ap * sc + s2 * ci * cc),
                     s2 * ap * sc - c2 * ci * cc])


def _wide_particles(rng, P: int, T: float) -> np.ndarray:
    tc = rng.uniform(T, T + TC_SPAN_YR * YEAR_S, P)
    mc = rng.uniform(*MC_RANGE, P)
    eta = rng.uniform(*ETA_RANGE, P)
    ct = rng.uniform(-1.0, 1.0, P)
    phi = rng.uniform(0.0, 2.0 * np.pi, P)
    e0 = rng.uniform(*E0_RANGE, P)
    return np.stack([tc, mc, eta, np.arccos(ct), phi, e0], axis=1)


def paper_range_particles(P: int, seed: int = 105) -> np.ndarray:
    """[P][6] particles uniform over the PAPER's own search ranges (PAPER.md:249-256 Table I, :313-325 Table III):
    t_c 3.3-3.8 yr, M_c 20-80 Msun, delta_mu 0-0.9 (eta = (1 - delta_mu^2)/4, reading A18), theta 0-pi, phi 0-2pi,
    e0 0-0.05.  BASELINE.json's configs use narrower masses and a wider t_c / e0 (reading A22); this population
    checks the stride selection where the paper itself searches."""
    rng = np.random.default_rng(seed)
    tc = rng.uniform(3.3 * YEAR_S, 3.8 * YEAR_S, P)
    mc = rng.uniform(20.0, 80.0, P)
    dmu = rng.uniform(0.0, 0.9, P)
    th = rng.uniform(0.0, np.pi, P)
    phi = rng.uniform(0.0, 2.0 * np.pi, P)
    e0 = rng.uniform(0.0, 0.05, P)
    return np.stack([tc, mc, 0.25 * (1.0 - dmu * dmu), th, phi, e0], axis=1)


def draw_particles(cfg: Config, P: Optional[int] = None) -> np.ndarray:
    """[P][6] float64 intrinsic parameters (tc, Mc, eta, theta, phi, e0) of config ``cfg``."""
    P = int(cfg.P[0] if P is None else P)
    rng = np.random.default_rng(cfg.particle_seed)
    inj = injection_params(cfg)
    if cfg.particle_rule == "wide":
        return _wide_particles(rng, P, cfg.T)
    if cfg.particle_rule == "swarms":
        # 8 independent swarms; each box = seeded centre +- 5% of the full range (10x shrink)
        n_sw = 8
        per = P // n_sw
        full = np.array([TC_SPAN_YR * YEAR_S, MC_RANGE[1] - MC_RANGE[0], ETA_RANGE[1] - ETA_RANGE[0],
                         2.0, 2.0 * np.pi, E0_RANGE[1] - E0_RANGE[0]])
        inj_u = inj.copy()
        inj_u[3] = math.cos(inj[3])                       # box is uniform in cos(theta)
        out = np.empty((n_sw * per, 6))
        for s in range(n_sw):
            centre = inj_u + rng.uniform(-0.05, 0.05, 6) * full
            u = centre + rng.uniform(-0.05, 0.05, (per, 6)) * full
            u[:, 2] = np.clip(u[:, 2], 0.05, 0.25)
            u[:, 3] = np.clip(u[:, 3], -1.0, 1.0)
            u[:, 5] = np.clip(u[:, 5], 0.0, None)
            u[:, 3] = np.arccos(u[:, 3])
            out[s * per:(s + 1) * per] = u
        return out
    if cfg.particle_rule == "bands":
        out = _wide_particles(rng, P, cfg.T)
        out[:, 0] = rng.uniform(1.0 * YEAR_S, 3.0 * YEAR_S, P)
        return out
    if cfg.particle_rule == "final":
        deg = math.pi / 180.0
        tc = inj[0] + rng.uniform(-1000.0, 1000.0, P)
        mc = inj[1] * (1.0 + rng.uniform(-1e-3, 1e-3, P))
        eta = rng.uniform(*ETA_RANGE, P)
        th = inj[3] + rng.uniform(-deg, deg, P)
        ph = inj[4] + rng.uniform(-deg, deg, P)
        e0 = np.clip(inj[5] + rng.uniform(-0.01, 0.01, P), 0.0, None)
        return np.stack([tc, mc, eta, th, ph, e0], axis=1)
    raise ValueError(cfg.particle_rule)


@dataclasses.dataclass
class Dataset:
    cfg: Config
    k_lo: int
    freq: np.ndarray          # [N] Hz
    sn: np.ndarray            # [N] one-sided PSD
    data: np.ndarray          # [N] complex128, noise (+ injection)
    dw: np.ndarray            # [N] complex128, data / S_n      (plan input)
    inv_sn: np.ndarray        # [N] float64, 1 / S_n            (plan input)
    injection: Optional[np.ndarray]   # [N] complex128 or None
    inj_params: np.ndarray    # [6]

    @property
    def n_bins(self) -> int:
        return int(self.freq.shape[0])

    @property
    def df(self) -> float:
        return 1.0 / self.cfg.T

    def edges(self, n_part: int) -> np.ndarray:
        return equal_bin_edges(self.n_bins, n_part)


TemplateFn = Callable[[np.ndarray, np.ndarray], Tuple[np.ndarray, np.ndarray]]


def make_dataset(cfg: Config, template_fn: Optional[TemplateFn] = None, noise: bool = True,
                 snr: Optional[float] = None, channel: str = "X") -> Dataset:
    """Noise (seeded) + injection.  ``template_fn(params6, freq) -> (u_plus, u_cross)`` supplies the
    two complex basis templates of the injection; ``None`` gives noise only.  The injection is
    h = (a1 + i a3) u_plus + (a2 + i a4) u_cross scaled so that 4 df sum |h|^2 / S_n = snr^2."""
    k_lo, n, f = frequency_grid(cfg.T, cfg.f_lo, cfg.f_hi)
    sn = psd_tdi(f, channel)                                # the TDI combination the data are in (default: the paper's X)
    d = coloured_noise(sn, cfg.T, cfg.noise_seed) if noise else np.zeros(n, dtype=np.complex128)
    inj = None
    pinj = injection_params(cfg)
    if template_fn is not None:
        up, uc = template_fn(pinj, f)
        a = injection_amplitudes()
        h = (a[0] + 1j * a[2]) * np.asarray(up) + (a[1] + 1j * a[3]) * np.asarray(uc)
        rho2 = 4.0 / cfg.T * float(np.sum((h.real ** 2 + h.imag ** 2) / sn))
        target = _INJ["snr"] if snr is None else snr
        inj = h * (target / math.sqrt(rho2))
        d = d + inj
    return Dataset(cfg, k_lo, f, sn, d, d / sn, 1.0 / sn, inj, pinj)
