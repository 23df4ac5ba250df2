"""Pins of the oracle's row-f2 functions (the paper's own segment limits): `template_band`,
`band_edges`, `fstat_bands`.  CPU only.  Each pin ties them to something other than themselves: a
textbook series the oracle does not contain, a time-domain simulation, hand-computed integers, the
zero-noise identity 2F = <h, h>."""
import math

import numpy as np
import pytest
from scipy import optimize

import synthetic.lisa_data as syn
import td_sim

YR = syn.YEAR_S
GMSUN = 4.925490947641267e-6


@pytest.fixture(scope="module")
def bands(orc):
    return syn.make_dataset(syn.BANDS_SMALL, orc.template)


def _ip(a, b, sn, df):
    """<a, b> = 4 df Re sum a conj(b) / S_n, retyped from PAPER.md:66 Eq. 4 (rectangle rule)."""
    return 4.0 * df * float(np.sum((a * np.conj(b)).real / sn))


def _tau_2pn(f, Mc, eta):
    """Time to coalescence from GW frequency f, circular orbit, to 2PN (the textbook series, e.g. Blanchet's
    review / Maggiore Eq. 5.266 extended): tau = (5/256) Mc^(-5/3) (pi f)^(-8/3) [1 + (4/3)(743/336 + 11 eta/4) x
    - (32 pi/5) x^(3/2) + 2 (3058673/1016064 + 5429 eta/1008 + 617 eta^2/144) x^2], x = (pi M f)^(2/3).
    The oracle never evaluates this series: it differentiates the phase of Eq. A3."""
    Mcs = Mc * GMSUN
    x = (math.pi * Mcs * eta ** -0.6 * f) ** (2.0 / 3.0)
    return (5.0 / 256.0) * Mcs ** (-5.0 / 3.0) * (math.pi * f) ** (-8.0 / 3.0) * (
        1.0 + (4.0 / 3.0) * (743.0 / 336.0 + 11.0 * eta / 4.0) * x - (32.0 * math.pi / 5.0) * x ** 1.5
        + 2.0 * (3058673.0 / 1016064.0 + 5429.0 * eta / 1008.0 + 617.0 * eta ** 2 / 144.0) * x * x)


def test_band_limits_match_the_textbook_time_to_coalescence(orc, bands):
    """the outer limits are the instantaneous frequencies at t = 0 and t = T.  For e_0 = 0 the
    frequency reached at time t solves tau(f) = t_c - t with the textbook 2PN series (the 2.5PN and 3PN terms
    the oracle also carries move it by 2e-6 of tau: a fraction of a bin here)."""
    ds = bands
    T = ds.cfg.T
    n_checked = 0
    for par in syn.draw_particles(ds.cfg)[:24]:
        par = par.copy()
        par[5] = 0.0
        k_lo, k_hi = orc.template_band(par, ds.freq, T)
        for t_obs, k in ((0.0, k_lo), (T, k_hi)):
            if k == 0 or k == ds.n_bins:
                continue                                  # the limit lies outside the grid
            f_t = optimize.brentq(lambda f: _tau_2pn(f, par[1], par[2]) - (par[0] - t_obs), 1e-3, 1.0, xtol=1e-16)
            # bin k is the first one at or past f_t
            assert abs((ds.k_lo + k) - f_t * T) <= 2.0
            n_checked += 1
    assert n_checked >= 10


def test_band_brackets_the_observation(orc, bands):
    """k_lo / k_hi against t_f itself (pinned by P6): t_f < 0 just below the band, 0 <= t_f <= T inside it,
    t_f > T just above."""
    ds = bands
    T = ds.cfg.T
    for par in syn.draw_particles(ds.cfg)[:32]:
        k_lo, k_hi = orc.template_band(par, ds.freq, T)
        assert 0 <= k_lo <= k_hi <= ds.n_bins
        tf = lambda k: orc.phase(par, ds.freq[k])[1]
        if k_lo > 0:
            assert tf(k_lo - 1) < 0.0
        if k_lo < ds.n_bins:
            assert tf(k_lo) >= 0.0
        if k_hi > 0:
            assert tf(k_hi - 1) <= T
        if k_hi < ds.n_bins:
            assert tf(k_hi) > T


def test_band_holds_the_power_of_a_time_domain_signal(orc):
    """A signal simulated in the TIME domain over [0, T] (tests/td_sim.py: Keplerian orbits, explicit links and
    TDI delays, no stationary-phase step) has its power between f(t = 0) and f(t = T): the band the oracle
    derives from t_f holds > 98 % of it, and the same band shifted by 15 % of its width loses > 7 %."""
    L = 2.5e9
    par = np.array([1.6 * YR, 40.0, 0.24, 1.1, 2.3, 0.03])
    dt, N = 16.0, 2 ** 19
    T = N * dt
    fg = np.linspace(0.015, 0.03, 12001)
    pt = np.array([orc.phase(par, f) for f in fg])
    sel = (pt[:, 1] > -0.03 * YR) & (pt[:, 1] < T + 0.03 * YR)
    chirp = td_sim.Chirp(fg[sel], pt[sel, 0], pt[sel, 1])
    cp, cc = 0.8 * np.exp(0.3j), 0.5 * np.exp(-1.1j)
    x = td_sim.tdi_x_time_domain(np.arange(N) * dt, chirp, cp, cc, par[3], par[4], L)
    power = np.abs(np.fft.rfft(x)) ** 2
    k0, k1 = int(0.015 * T), int(0.03 * T)
    fk = np.arange(k0, k1) / T
    k_lo, k_hi = orc.template_band(par, fk, T)
    assert 0 < k_lo < k_hi < fk.shape[0]
    total = power[k0:k1].sum()
    assert power.sum() == pytest.approx(total, rel=2e-2)              # nothing outside 15-30 mHz anyway
    inside = power[k0 + k_lo:k0 + k_hi].sum()
    assert inside > 0.98 * total
    sh = int(0.15 * (k_hi - k_lo))
    assert power[k0 + k_lo + sh:k0 + k_hi + sh].sum() < 0.93 * total
    assert power[k0 + k_lo - sh:k0 + k_hi - sh].sum() < 0.93 * total


def test_band_edges_hand_computed(orc):
    """Reading A26 on integers worked out by hand."""
    np.testing.assert_array_equal(orc.band_edges(3, 13, 100, 4, 1), [3, 5, 8, 10, 13])
    # lattice 4: (3 + 2) // 4 = 1, (13 + 2) // 4 = 3: two cells for four partitions, two of them empty
    np.testing.assert_array_equal(orc.band_edges(3, 13, 100, 4, 4), [4, 4, 8, 8, 12])
    # rounding half up, and clipping of the last edge to the grid
    np.testing.assert_array_equal(orc.band_edges(4, 100, 100, 2, 8), [8, 56, 100])
    np.testing.assert_array_equal(orc.band_edges(0, 0, 100, 3, 1), [0, 0, 0, 0])
    np.testing.assert_array_equal(orc.band_edges(100, 100, 100, 3, 16), [96, 96, 96, 96])
    np.testing.assert_array_equal(orc.band_edges(0, 7, 7, 7, 1), np.arange(8))


def test_band_edges_properties(orc):
    rng = np.random.default_rng(3)
    for _ in range(300):
        n = int(rng.integers(1, 5000))
        lo, hi = np.sort(rng.integers(0, n + 1, 2))
        n_seg = int(rng.integers(1, 40))
        Cc = int(rng.choice([1, 2, 8, 64, 128]))
        e = orc.band_edges(lo, hi, n, n_seg, Cc)
        assert e.shape == (n_seg + 1,) and np.all(np.diff(e) >= 0) and e[0] >= 0 and e[-1] <= n
        assert abs(e[0] - lo) <= Cc // 2 + (Cc if e[0] == n else 0) and abs(e[-1] - hi) <= Cc // 2
        inner = e[(e % Cc != 0)]
        assert np.all(inner == n)                         # every edge sits on the lattice, or at the grid's end
        d = np.diff(e)
        if e[-1] < n:
            assert d.max() - d.min() <= Cc                # equal parts up to one lattice cell


@pytest.mark.parametrize("n_seg", [1, 4, 16])
def test_zero_noise_recovers_the_in_band_snr(orc, n_seg):
    """Data = the injection windowed to its own band, no noise: every partition recovers its share,
    2 F_k = <h, h>_k (Eq. 7 at a = the injected amplitudes), so 2 F = rho^2 in band."""
    ds = syn.make_dataset(syn.BANDS_SMALL, orc.template, noise=False)
    par = ds.inj_params
    k_lo, k_hi = orc.template_band(par, ds.freq, ds.cfg.T)
    assert 0 < k_lo < k_hi < ds.n_bins
    h = np.zeros_like(ds.injection)
    h[k_lo:k_hi] = ds.injection[k_lo:k_hi]
    F, Fk, edges = orc.fstat_bands(ds.freq, h / ds.sn, ds.inv_sn, par[None, :], n_seg, 1)
    assert edges[0, 0] == k_lo and edges[0, -1] == k_hi
    for j in range(n_seg):
        sl = slice(edges[0, j], edges[0, j + 1])
        assert 2.0 * Fk[0, j] == pytest.approx(_ip(h[sl], h[sl], ds.sn[sl], ds.df), rel=1e-9)
    assert 2.0 * F[0] == pytest.approx(_ip(h, h, ds.sn, ds.df), rel=1e-9)
    # the part of the injection outside the band is not seen at all
    F2, _, _ = orc.fstat_bands(ds.freq, ds.injection / ds.sn, ds.inv_sn, par[None, :], n_seg, 1)
    assert F2[0] == pytest.approx(F[0], rel=1e-12)


def test_bands_reduce_to_fixed_edges_on_the_band(orc, bands):
    """With the band's own bins as the grid, row f2 is the fixed-edge statistic (`fstat_batch`, pins P1-P5)
    with equal-bin partitions."""
    ds = bands
    par = syn.draw_particles(ds.cfg)
    done = 0
    for p in par[:20]:
        k_lo, k_hi = orc.template_band(p, ds.freq, ds.cfg.T)
        if k_hi - k_lo < 64:
            continue
        F, Fk, edges = orc.fstat_bands(ds.freq, ds.dw, ds.inv_sn, p[None, :], 4, 1)
        sl = slice(k_lo, k_hi)
        Fr, Fkr = orc.fstat_batch(ds.freq[sl], ds.dw[sl], ds.inv_sn[sl], syn.equal_bin_edges(k_hi - k_lo, 4), p[None, :])
        np.testing.assert_array_equal(edges[0] - k_lo, syn.equal_bin_edges(k_hi - k_lo, 4))
        np.testing.assert_allclose(Fk, Fkr, rtol=1e-9)
        assert F[0] == pytest.approx(Fr[0], rel=1e-9)
        done += 1
    assert done >= 5


def test_bands_invalid_and_empty(orc, bands):
    ds = bands
    par = syn.draw_particles(ds.cfg)[:4].copy()
    par[1, 1] = -1.0
    par[2, 0] = 0.2 * YR                                   # merges long before f reaches 20 mHz... band above the grid
    F, Fk, edges = orc.fstat_bands(ds.freq, ds.dw, ds.inv_sn, par, 4, 64)
    assert np.isneginf(F[1]) and np.all(np.isneginf(Fk[1]))
    k_lo, k_hi = orc.template_band(par[2], ds.freq, ds.cfg.T)
    if k_hi == k_lo:
        assert F[2] == 0.0 and np.all(Fk[2] == 0.0)
