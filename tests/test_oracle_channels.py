"""Pins of the oracle's row-f4 function `fstat_batch_channels` (Eq. 3: the sum over TDI
combinations with mutually independent noise).  CPU only."""
import math

import numpy as np
import pytest
from scipy import optimize

import synthetic.lisa_data as syn

LAM = 2.0 * math.pi / 3.0


def _ip(a, b, sn, df):
    """<a, b> = 4 df Re sum a conj(b) / S_n, retyped from PAPER.md:66 Eq. 4 (rectangle rule)."""
    return 4.0 * df * float(np.sum((a * np.conj(b)).real / sn))


def _channel_opts(orc, n):
    return [orc.default_options(orbit_lambda=c * LAM) for c in range(n)]


def test_lambda_shift_relabels_the_spacecraft(orc):
    """Reading A9: beta_n = 2 pi n / 3 + lambda, so lambda + 2 pi/3 moves spacecraft 2 -> 1, 3 -> 2, 1 -> 3: the X
    combination of the shifted constellation (centred on "1", arms to "2" and "3") is Y of the original one (centred
    on 2, arms to 3 and 1), and once more gives Z."""
    for t in (0.0, 1.234e7, 6.1e7):
        p0 = orc.orbit(t)
        p1 = orc.orbit(t, orc.default_options(orbit_lambda=LAM))
        p2 = orc.orbit(t, orc.default_options(orbit_lambda=2 * LAM))
        np.testing.assert_allclose(p1, np.roll(p0, -1, axis=0), rtol=0, atol=1e-3)
        np.testing.assert_allclose(p2, np.roll(p0, -2, axis=0), rtol=0, atol=1e-3)


def _three_channel_data(orc, noise=True, snr=12.0):
    cfg = syn.CONFIGS[0]
    k_lo, n, f = syn.frequency_grid(cfg.T, cfg.f_lo, cfg.f_hi)
    sn = syn.psd_tdi_x(f)                                  # equal arms: X, Y, Z share the PSD
    opts = _channel_opts(orc, 3)
    inj = syn.injection_params(cfg)
    a = syn.injection_amplitudes()
    hs = []
    for o in opts:
        up, uc = orc.template(inj, f, o)
        hs.append((a[0] + 1j * a[2]) * up + (a[1] + 1j * a[3]) * uc)
    rho2 = sum(_ip(h, h, sn, 1.0 / cfg.T) for h in hs)
    scale = snr / math.sqrt(rho2)                          # ONE amplitude vector for all channels
    data = [h * scale + (syn.coloured_noise(sn, cfg.T, 40 + c) if noise else 0.0) for c, h in enumerate(hs)]
    return cfg, f, sn, opts, inj, data, [h * scale for h in hs]


def test_channels_equal_bruteforce_maximum_of_eq3(orc):
    """F_k = max over the four COMMON amplitudes of sum_I [<d_I, h_I> - <h_I, h_I>/2] (Eq. 3), found by numerical
    maximisation from several starts, never via N, M or a linear solve."""
    cfg, f, sn, opts, inj, data, _ = _three_channel_data(orc)
    df = 1.0 / cfg.T
    edges = syn.equal_bin_edges(f.shape[0], 4)
    par = syn.draw_particles(cfg)[:2]
    chans = [(d / sn, 1.0 / sn, o) for d, o in zip(data[:2], opts[:2])]            # two channels
    F, Fk = orc.fstat_batch_channels(f, chans, edges, par)
    rng = np.random.default_rng(11)
    for p in range(par.shape[0]):
        tmpl = [orc.template(par[p], f, o) for o in opts[:2]]
        for j in range(4):
            sl = slice(edges[j], edges[j + 1])
            basis = [[up[sl], uc[sl], 1j * up[sl], 1j * uc[sl]] for up, uc in tmpl]
            scale = [1.0 / math.sqrt(sum(_ip(b[i], b[i], sn[sl], df) for b in basis)) for i in range(4)]

            def neg_lambda(x):
                tot = 0.0
                for c, b in enumerate(basis):
                    h = sum(x[i] * scale[i] * b[i] for i in range(4))
                    tot += _ip(data[c][sl], h, sn[sl], df) - 0.5 * _ip(h, h, sn[sl], df)
                return -tot

            best = min(optimize.minimize(neg_lambda, rng.standard_normal(4), method="BFGS",
                                         options={"gtol": 1e-10}).fun for _ in range(3))
            assert -best == pytest.approx(Fk[p, j], rel=1e-6)


@pytest.mark.parametrize("n_part", [1, 4])
def test_zero_noise_recovers_the_network_snr(orc, n_part):
    """One signal seen by X, Y, Z with the same four amplitudes, no noise, evaluated at its own parameters:
    2 F = sum_I <h_I, h_I> = 144; any single channel recovers only its own share."""
    cfg, f, sn, opts, inj, data, hs = _three_channel_data(orc, noise=False)
    df = 1.0 / cfg.T
    edges = syn.equal_bin_edges(f.shape[0], n_part)
    chans = [(d / sn, 1.0 / sn, o) for d, o in zip(data, opts)]
    F, Fk = orc.fstat_batch_channels(f, chans, edges, inj[None, :])
    assert 2.0 * F[0] == pytest.approx(144.0, rel=1e-9)
    for j in range(n_part):
        sl = slice(edges[j], edges[j + 1])
        assert 2.0 * Fk[0, j] == pytest.approx(sum(_ip(h[sl], h[sl], sn[sl], df) for h in hs), rel=1e-9)
    F1, _ = orc.fstat_batch(f, chans[0][0], chans[0][1], edges, inj[None, :], opts[0])
    assert 2.0 * F1[0] == pytest.approx(_ip(hs[0], hs[0], sn, df), rel=1e-9) and F1[0] < 0.6 * F[0]


def test_one_channel_is_the_single_channel_statistic_and_noise_stays_chi2(orc):
    cfg, f, sn, opts, inj, data, _ = _three_channel_data(orc, snr=0.0)
    edges = syn.equal_bin_edges(f.shape[0], 4)
    par = syn.draw_particles(cfg)
    chans = [(d / sn, 1.0 / sn, o) for d, o in zip(data, opts)]
    F1, Fk1 = orc.fstat_batch_channels(f, chans[:1], edges, par[:8])
    F0, Fk0 = orc.fstat_batch(f, chans[0][0], chans[0][1], edges, par[:8], opts[0])
    np.testing.assert_allclose(Fk1, Fk0, rtol=1e-12)
    # pure noise in three channels: 2 F_k is still chi^2 with 4 degrees of freedom (four common amplitudes)
    _, Fk3 = orc.fstat_batch_channels(f, chans, edges, par)
    m = 2.0 * Fk3.mean()
    assert 4.0 - 0.9 < m < 4.0 + 0.9                       # 256 correlated-ish draws: loose, a factor-of-N_I slip fails


# ----------------------------------------------------------------------------- P19: Y, Z, A, E, T responses
def _resp(orc, par, f, t, ch, **kw):
    return np.array(orc.response(par, f, t, orc.default_options(tdi_channel=orc.TDI_CHANNELS[ch], **kw)))


def test_p19_y_and_z_are_x_of_the_relabelled_constellation(orc):
    """Y and Z as the oracle builds them (Michelson centred on spacecraft 2, 3) equal the pinned X response of the
    constellation with its spacecraft relabelled cyclically (orbit_lambda + 2 pi/3, + 4 pi/3: P14)."""
    rng = np.random.default_rng(19)
    for _ in range(20):
        par = np.array([0.0, 30.0, 0.25, math.acos(rng.uniform(-1, 1)), rng.uniform(0, 2 * math.pi), 0.0])
        f, t, lam = rng.uniform(1e-3, 0.1), rng.uniform(0, 3 * syn.YEAR_S), rng.uniform(-1, 1)
        for ch, shift in (("Y", 2.0 * math.pi / 3.0), ("Z", 4.0 * math.pi / 3.0)):
            a = _resp(orc, par, f, t, ch, orbit_lambda=lam)
            b = _resp(orc, par, f, t, "X", orbit_lambda=lam + shift)
            assert np.max(np.abs(a - b)) <= 1e-12 * np.max(np.abs(b))


def test_p19_aet_are_the_combinations_of_ref_64(orc):
    """A = (Z - X)/sqrt 2, E = (X - 2Y + Z)/sqrt 6, T = (X + Y + Z)/sqrt 3 (reading A28), and the long-wavelength
    behaviour that makes T the 'null' channel: for f << c / (2 pi L) = 19 mHz the gravitational-wave response of
    X + Y + Z cancels at leading order."""
    par = np.array([0.0, 30.0, 0.25, 1.1, 2.3, 0.0])
    t = 0.37 * syn.YEAR_S
    ratio = {}
    for f in (1e-4, 1e-3, 2e-2):
        X, Y, Z = (_resp(orc, par, f, t, c) for c in "XYZ")
        A, E, T = (_resp(orc, par, f, t, c) for c in "AET")
        np.testing.assert_allclose(A, (Z - X) / math.sqrt(2.0), rtol=1e-13, atol=1e-16 * abs(X).max())
        np.testing.assert_allclose(E, (X - 2.0 * Y + Z) / math.sqrt(6.0), rtol=1e-13, atol=1e-16 * abs(X).max())
        np.testing.assert_allclose(T, (X + Y + Z) / math.sqrt(3.0), rtol=1e-13, atol=1e-14 * abs(X).max())
        ratio[f] = np.abs(T).max() / np.abs(A).max()
    # leading order cancels identically (xi is symmetric in the arm direction: sum_v [xi_(v,v+2) - xi_(v,v+1)] = 0),
    # so T / A falls at least like (f / 19 mHz)^2 towards low frequencies
    assert ratio[1e-4] < 1e-6 and ratio[1e-3] < 1e-3 and ratio[2e-2] > 1e-2
    assert ratio[1e-3] / ratio[1e-4] > 90.0


def test_p19_aet_frequency_domain_response_matches_time_domain_simulation(orc):
    """The P9 check for the A and E templates: X(t), Y(t), Z(t) simulated in the time domain (explicit link delays,
    Keplerian orbits, tests/td_sim.py), combined into A(t), E(t), T(t), Fourier transformed and compared as complex
    overlaps with x~(f) = T_I(f) h~(f) of Eq. 17.  T carries little signal below 30 mHz: its amplitude is checked
    instead of its phase-sensitive overlap to the same level."""
    import td_sim
    from scipy.signal.windows import tukey
    L = 2.5e9
    YR = syn.YEAR_S
    par = np.array([1.6 * YR, 40.0, 0.24, 1.1, 2.3, 0.03])
    dt, N = 16.0, 2 ** 20
    T_obs = N * dt
    fg = np.linspace(0.015, 0.03, 12001)
    pt = np.array([orc.phase(par, f) for f in fg])
    sel = (pt[:, 1] > -0.03 * YR) & (pt[:, 1] < T_obs + 0.03 * YR)
    chirp = td_sim.Chirp(fg[sel], pt[sel, 0], pt[sel, 1])
    cp, cc = 0.8 * np.exp(0.3j), 0.5 * np.exp(-1.1j)
    t = np.arange(N) * dt
    xyz = [td_sim.tdi_michelson_time_domain(t, chirp, cp, cc, par[3], par[4], L, v) for v in range(3)]
    td = {"A": (xyz[2] - xyz[0]) / math.sqrt(2.0), "E": (xyz[0] - 2.0 * xyz[1] + xyz[2]) / math.sqrt(6.0),
          "T": (xyz[0] + xyz[1] + xyz[2]) / math.sqrt(3.0)}
    fk = np.arange(N // 2 + 1) / T_obs
    tf_k = np.interp(fk, fg, pt[:, 1])
    band = (tf_k > 0.25 * T_obs) & (tf_k < 0.75 * T_obs)
    assert band.sum() > 20000
    power = {}
    for ch in "AET":
        X = (np.fft.rfft(td[ch] * tukey(N, 0.2)) * dt)[band]
        up, uc = orc.template(par, fk[band], orc.default_options(tdi_channel=orc.TDI_CHANNELS[ch]))
        Xfd = cp * up + cc * uc
        overlap = np.sum(X * np.conj(Xfd)) / math.sqrt(np.sum(abs(X) ** 2) * np.sum(abs(Xfd) ** 2))
        power[ch] = (np.sum(abs(X) ** 2), np.sum(abs(Xfd) ** 2))
        if ch in "AE":
            assert overlap.real > 0.999 and abs(overlap.imag) < 0.03, (ch, overlap)
        assert math.sqrt(power[ch][0] / power[ch][1]) == pytest.approx(1.0, abs=2e-2), ch
    assert power["T"][1] < 0.2 * power["A"][1]


def test_p19_aet_channel_sum_recovers_the_network_snr(orc):
    """Zero noise, one signal seen in A, E and T with one amplitude vector: 2F over the three channels = the sum of
    the three <h_I, h_I> (Eq. 3 :62); a single channel recovers only its share."""
    cfg = syn.CONFIGS[0]
    _, n, f = syn.frequency_grid(cfg.T, cfg.f_lo, cfg.f_hi)
    par = syn.injection_params(cfg)
    a = syn.injection_amplitudes()
    edges = syn.equal_bin_edges(n, 4)
    df = 1.0 / cfg.T
    chans, snr2 = [], 0.0
    sn = syn.psd_tdi_x(f)                                   # any positive weight will do for this identity
    for ch in "AET":
        o = orc.default_options(tdi_channel=orc.TDI_CHANNELS[ch])
        up, uc = orc.template(par, f, o)
        h = (a[0] + 1j * a[2]) * up + (a[1] + 1j * a[3]) * uc
        snr2 += 4.0 * df * float(np.sum(np.abs(h) ** 2 / sn))
        chans.append((h / sn, 1.0 / sn, o))
    F, Fk = orc.fstat_batch_channels(f, chans, edges, par[None, :])
    assert 2.0 * F[0] == pytest.approx(snr2, rel=1e-9)
    F1, _ = orc.fstat_batch_channels(f, chans[:1], edges, par[None, :])
    assert 0.0 < 2.0 * F1[0] < 0.9 * snr2
