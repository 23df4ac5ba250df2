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
