"""extrinsic amplitudes a = M^-1 N (Eq. 10) from the library against the oracle's
4x4 solve, and the recovery of (D_L, iota, psi, phi_c) by Eq. B2-B3 (:426-440): the library's host function
fstat_extrinsic_from_amplitudes (through the C ABI) against the oracle's plain restatement of App. B
(oracle/extrinsic_oracle.py), both pinned by the round trip through Eq. B1 (:413-420, retyped here)."""
import math

import numpy as np
import pytest

import synthetic as syn
from oracle import extrinsic_oracle as xo
from paper_2407_10797_b200 import build as _cuda_build
from paper_2407_10797_b200.extrinsic import amplitudes_from_extrinsic, extrinsic_from_amplitudes

_cuda_build.build()                                       # host functions of the C-ABI library: no GPU needed


def _b1(d_l, psi, iota, phi_c):
    """Eq. B1 as printed (:413-420)."""
    p = (1.0 + math.cos(iota) ** 2) / 2.0
    a1 = (math.cos(2 * psi) * p * math.cos(phi_c) - math.sin(2 * psi) * math.cos(iota) * math.sin(phi_c)) / d_l
    a2 = -(math.sin(2 * psi) * p * math.cos(phi_c) + math.cos(2 * psi) * math.cos(iota) * math.sin(phi_c)) / d_l
    a3 = -(math.cos(2 * psi) * p * math.sin(phi_c) + math.sin(2 * psi) * math.cos(iota) * math.cos(phi_c)) / d_l
    a4 = (math.sin(2 * psi) * p * math.sin(phi_c) - math.cos(2 * psi) * math.cos(iota) * math.cos(phi_c)) / d_l
    return np.array([a1, a2, a3, a4])


def test_b2_b3_invert_b1_inside_the_principal_branches():
    rng = np.random.default_rng(7)
    for _ in range(200):
        d_l, psi = rng.uniform(0.3, 5.0), rng.uniform(-math.pi / 4, math.pi / 4)
        iota, phi_c = rng.uniform(0.0, math.pi), rng.uniform(-math.pi / 2, math.pi / 2)
        r = extrinsic_from_amplitudes(_b1(d_l, psi, iota, phi_c))
        assert r["D_L"] == pytest.approx(d_l, rel=1e-10)
        assert r["iota"] == pytest.approx(iota, abs=2e-6 / max(math.sin(iota), 1e-3))
        # psi and phi_c become degenerate (only psi +- phi_c is fixed) as the orbit turns face-on
        tol = 1e-7 / max(1.0 - abs(math.cos(iota)), 1e-3)
        assert r["psi"] == pytest.approx(psi, abs=tol)
        assert r["phi_c"] == pytest.approx(phi_c, abs=tol)
        np.testing.assert_allclose(_b1(r["D_L"], r["psi"], r["iota"], r["phi_c"]), _b1(d_l, psi, iota, phi_c),
                                   rtol=0, atol=1e-7 / d_l)      # iota loses half the digits near face-on
        np.testing.assert_allclose(amplitudes_from_extrinsic(d_l, psi, iota, phi_c), _b1(d_l, psi, iota, phi_c),
                                   rtol=0, atol=1e-15)


def test_outside_the_principal_branches_the_recovered_set_reproduces_the_amplitudes():
    """psi and phi_c are only defined up to the discrete symmetries of Eq. B1; whatever branch Eq. B2 picks,
    feeding it back through Eq. B1 must give the same four amplitudes (Table I's psi = 1.2501 is outside)."""
    rng = np.random.default_rng(8)
    for _ in range(200):
        d_l, psi = rng.uniform(0.3, 5.0), rng.uniform(-math.pi, math.pi)
        iota, phi_c = rng.uniform(0.0, math.pi), rng.uniform(-math.pi, math.pi)
        a = _b1(d_l, psi, iota, phi_c)
        r = extrinsic_from_amplitudes(a)
        # psi and phi_c come from two separate arctans and lose digits as the orbit turns face-on
        tol = 1e-8 / (d_l * max(1.0 - abs(math.cos(iota)), 1e-4))
        np.testing.assert_allclose(_b1(r["D_L"], r["psi"], r["iota"], r["phi_c"]), a, rtol=0, atol=tol)
        assert r["D_L"] == pytest.approx(d_l, rel=1e-10) and r["iota"] == pytest.approx(iota, abs=2e-6 / max(math.sin(iota), 1e-3))


def test_oracle_b2_b3_inverts_b1_and_the_library_agrees_with_it():
    """The oracle's App. B (Eq. B2-B3 as printed + reading A25) is pinned by the round trip through Eq. B1 as printed;
    the library's C function, called through the ABI, gives the oracle's four numbers on random amplitude vectors."""
    rng = np.random.default_rng(9)
    for _ in range(300):
        d_l, psi = rng.uniform(0.3, 5.0), rng.uniform(-math.pi, math.pi)
        iota, phi_c = rng.uniform(0.0, math.pi), rng.uniform(-math.pi, math.pi)
        a = _b1(d_l, psi, iota, phi_c)
        np.testing.assert_allclose(xo.b1(d_l, psi, iota, phi_c), a, rtol=0, atol=1e-15)
        o = xo.b2_b3(a)
        assert o[0] == pytest.approx(d_l, rel=1e-7) and o[1] == pytest.approx(iota, abs=2e-6 / max(math.sin(iota), 1e-3))
        tol = 1e-8 / (d_l * max(1.0 - abs(math.cos(iota)), 1e-4))
        np.testing.assert_allclose(_b1(*[o[0], o[2], o[1], o[3]]), a, rtol=0, atol=max(tol, 1e-7 / d_l))
        r = extrinsic_from_amplitudes(a)
        near_face_on = max(1.0 - abs(math.cos(iota)), 1e-4)
        assert r["D_L"] == pytest.approx(o[0], rel=1e-6)      # the oracle keeps the printed sqrt(A_+^2 - A_x^2): cancellation
        assert r["iota"] == pytest.approx(o[1], abs=1e-5 / max(math.sin(iota), 1e-3))
        assert r["psi"] == pytest.approx(o[2], abs=1e-6 / near_face_on)
        assert abs(math.remainder(r["phi_c"] - o[3], 2.0 * math.pi)) <= 1e-6 / near_face_on
    with pytest.raises(Exception):
        extrinsic_from_amplitudes([np.nan, 0.0, 0.0, 0.0])
    assert extrinsic_from_amplitudes([0.0, 0.0, 0.0, 0.0])["D_L"] == math.inf


def test_amplitude_constant_restores_metres():
    mc, d_l_m = 30.0, 3.0e24                                   # ~100 Mpc
    k = -math.sqrt(5 / 24) * (30 * 4.925490947641267e-6) ** (5 / 6) / math.pi ** (2 / 3)      # Eq. A2 (:402) without 1/D_L
    a_lib = k * _b1(d_l_m / 299792458.0, 0.3, 1.0, -0.4)
    r = extrinsic_from_amplitudes(a_lib, chirp_mass_msun=mc)
    assert r["D_L"] == pytest.approx(d_l_m, rel=1e-10) and r["iota"] == pytest.approx(1.0, abs=1e-8)


def test_p20_physical_time_domain_binary_recovers_distance_and_inclination(orc):
    """Pin P20 (nothing independent pinned the absolute normalisation behind D_L).  The injection is PHYSICAL
    and carries nothing of App. A-B: the quadrupole-formula strain of two point masses on a circular orbit at a known
    distance, with a known orbital angular momentum direction (tests/td_sim.py PhysicalBinary), through four explicit
    one-way links on Keplerian orbits and explicit TDI delays, FFT.  The oracle's amplitudes a = M^-1 N of that data
    (white noise weights, no noise) go through Eq. B2-B3 (oracle restatement) and through the library's host function
    fstat_extrinsic_from_amplitudes with the Eq. A2 constant restored.  Recovered: D_L within 5 %, iota within 0.05 rad
    -- the size of error the paper's own N = 0 response leaves (match > 0.999, is an amplitude residual of up
    to 4.5 %) -- which rules out a factor 2, sqrt 2 or a dropped 1/2 anywhere in the link factor, the TDI factor, Eq. A2's
    constant or Eq. B1-B3.  It also fixes what the angles mean physically (reading A31): iota is the angle between the
    orbital angular momentum and the propagation direction k (source -> observer); psi = pi/2 - (angle of Lhat's sky
    projection from u towards v), modulo pi/2; advancing the orbital phase by dPhi/2 lowers phi_c by dPhi."""
    import sys
    import os
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    import td_sim
    from scipy.signal.windows import tukey
    year, c_light, gms = 31557600.0, 299792458.0, 4.925490947641267e-6
    L = 2.5e9
    par = np.array([1.6 * year, 40.0, 0.24, 1.1, 2.3, 0.0])
    dt, N = 16.0, 2 ** 20
    T = N * dt
    fg = np.linspace(0.015, 0.03, 12001)
    pt = np.array([orc.phase(par, f) for f in fg])
    sel = (pt[:, 1] > -0.03 * year) & (pt[:, 1] < T + 0.03 * year)
    chirp = td_sim.Chirp(fg[sel], pt[sel, 0], pt[sel, 1])
    k, u, v = orc.sky_basis(par[3], par[4])
    # (D_L [m], iota, pol, phi0): near face-on, the same with the orbital phase advanced, retrograde, near edge-on
    sets = [(3.0e24, 0.6, 0.3, 0.0), (3.0e24, 0.6, 0.3, 1.0), (1.0e25, 2.2, -0.5, 0.4), (3.0e24, 1.2, 1.3, 0.0)]
    src = td_sim.PhysicalBinary(chirp, par[1] * gms, np.asarray(k), np.asarray(u), np.asarray(v),
                                [(d / c_light, i, p, f0) for d, i, p, f0 in sets])
    t = np.arange(N) * dt
    x = td_sim.tdi_michelson_time_domain(t, src, None, None, par[3], par[4], L, 0)          # [n_sets][N]
    X = np.fft.rfft(x * tukey(N, 0.2)[None, :], axis=1) * dt
    fk = np.arange(N // 2 + 1) / T
    tf_k = np.interp(fk, fg, pt[:, 1])
    band = np.nonzero((tf_k > 0.25 * T) & (tf_k < 0.75 * T))[0]
    lo, hi = int(band[0]), int(band[-1]) + 1
    up, uc = orc.template(par, fk[lo:hi])
    w = np.ones(hi - lo)
    K = -math.sqrt(5.0 / 24.0) * (par[1] * gms) ** (5.0 / 6.0) / math.pi ** (2.0 / 3.0)       # Eq. A2 (:402) without 1/D_L
    rec = []
    for n, (d_m, iota, pol, phi0) in enumerate(sets):
        _, a, flag = orc.fstat_partition(X[n, lo:hi], w, up, uc, 1.0 / T, 0, hi - lo, 2)
        assert flag == 0
        d_s, io, ps, pc = xo.b2_b3(a / K)                                                       # oracle App. B
        r = extrinsic_from_amplitudes(a, chirp_mass_msun=par[1])                               # library host function
        assert r["D_L"] == pytest.approx(d_s * c_light, rel=1e-9) and r["iota"] == pytest.approx(io, abs=1e-9)
        assert r["D_L"] == pytest.approx(d_m, rel=0.05), (n, r["D_L"] / d_m)
        assert io == pytest.approx(iota, abs=0.05), n
        rec.append((ps, pc))
        if 1.0 < iota < 2.3:                               # psi is defined only away from face-on
            dpsi = (ps - (math.pi / 2.0 - pol) + math.pi / 4.0) % (math.pi / 2.0) - math.pi / 4.0
            assert abs(dpsi) < 0.1, (n, ps, pol)
    dphi = (rec[1][1] - rec[0][1] + 1.0 + math.pi) % (2.0 * math.pi) - math.pi                 # phi_c moved by -phi0
    assert abs(dphi) < 1e-6 and rec[1][0] == pytest.approx(rec[0][0], abs=1e-6)


@pytest.mark.gpu
def test_amplitudes_match_the_oracle_and_recover_the_injection(orc):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2407_10797_b200 as fs
    year = 31557600.0
    cfg = syn.Config(14, "amp_slice", 2.5 * year, 0.0200, 0.0201, (4,), (40,), 3.5 * year, "wide")
    # (i) noisy data, N_p = 4: a = M^-1 N of every partition against the oracle's 4x4 Cholesky solve
    ds = syn.make_dataset(cfg, orc.template)
    par = syn.draw_particles(cfg)
    edges = ds.edges(4)
    _, _, NM, flags = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par, want_NM=True)
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges) as plan:
        amp = fs.fstat_eval_amplitudes(plan, torch.as_tensor(par, device="cuda")).cpu().numpy()
        F, Fk = fs.fstat_eval_batch(plan, torch.as_tensor(par, device="cuda"))
        Fk = Fk.cpu().numpy()
    assert amp.shape == (par.shape[0], 4, 4)
    for p in range(par.shape[0]):
        for k in range(4):
            N, M = NM[p, k, :4], NM[p, k, 4:].reshape(4, 4)
            F_o, a_o, _ = orc.fstat_from_NM(N, M)
            assert np.linalg.norm(amp[p, k] - a_o) <= 1e-5 * np.linalg.norm(a_o)
            assert 0.5 * amp[p, k] @ N == pytest.approx(Fk[p, k], rel=1e-6)       # F = a.N / 2 at the maximum
    # (ii) zero noise, N_p = 1, at the injected parameters: the amplitudes are the injected ones (times the
    # SNR normalisation), and Eq. B2-B3 give back an extrinsic set that reproduces them
    ds0 = syn.make_dataset(cfg, orc.template, noise=False)
    a_inj = syn.injection_amplitudes()
    with fs.fstat_plan_create(ds0.freq, ds0.dw, ds0.inv_sn, ds0.edges(1)) as plan:
        a0 = fs.fstat_eval_amplitudes(plan, torch.as_tensor(ds0.inj_params[None, :], device="cuda")).cpu().numpy()[0, 0]
    scale = float(a0 @ a_inj / (a_inj @ a_inj))
    assert scale > 0.0
    np.testing.assert_allclose(a0, scale * a_inj, rtol=0, atol=1e-8 * np.linalg.norm(a0))
    r = extrinsic_from_amplitudes(a0)
    np.testing.assert_allclose(_b1(r["D_L"], r["psi"], r["iota"], r["phi_c"]), a0, rtol=0, atol=1e-8 * np.linalg.norm(a0))
    assert r["iota"] == pytest.approx(0.5329, abs=1e-6)        # Table I (:257): the injected inclination


@pytest.mark.gpu
@pytest.mark.parametrize("n_seg,lattice", [(1, 1), (4, 1), (4, 64)])
def test_band_amplitudes_match_the_oracle_and_recover_the_injection(orc, n_seg, lattice):
    """Rows f2 x f3: the amplitudes of every partition of every template's own band (fstat_eval_amplitudes_bands)
    against the oracle's 4x4 solve over the same bins; and, zero noise at the injected parameters, the coherent
    estimate over the band gives back the injected amplitudes and Table I's inclination."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2407_10797_b200 as fs
    cfg = syn.BANDS_SMALL
    ds = syn.make_dataset(cfg, orc.template)
    par = syn.draw_particles(cfg)[:32].copy()
    par[3, 2] = 0.3                                          # invalid: NaN amplitudes
    F_o, Fk_o, edges, a_o = orc.fstat_bands(ds.freq, ds.dw, ds.inv_sn, par, n_seg, lattice, want_amp=True)
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(1)) as plan:
        amp = fs.fstat_eval_amplitudes_bands(plan, torch.as_tensor(par, device="cuda"), n_seg, lattice).cpu().numpy()
    assert amp.shape == (32, n_seg, 4) and np.all(np.isnan(amp[3])) and np.all(np.isnan(a_o[3]))
    n_live = 0
    for p in range(32):
        if p == 3:
            continue
        for k in range(n_seg):
            if edges[p, k + 1] > edges[p, k]:
                assert np.linalg.norm(amp[p, k] - a_o[p, k]) <= 1e-5 * np.linalg.norm(a_o[p, k])
                n_live += 1
            else:
                assert np.all(amp[p, k] == 0.0)
    assert n_live >= 15 * n_seg
    if n_seg == 1:
        ds0 = syn.make_dataset(cfg, orc.template, noise=False)
        a_inj = syn.injection_amplitudes()
        with fs.fstat_plan_create(ds0.freq, ds0.dw, ds0.inv_sn, ds0.edges(1)) as plan:
            a0 = fs.fstat_eval_amplitudes_bands(plan, torch.as_tensor(ds0.inj_params[None, :], device="cuda"), 1,
                                                lattice).cpu().numpy()[0, 0]
        scale = float(a0 @ a_inj / (a_inj @ a_inj))
        assert scale > 0.0
        np.testing.assert_allclose(a0, scale * a_inj, rtol=0, atol=1e-8 * np.linalg.norm(a0))
        assert extrinsic_from_amplitudes(a0)["iota"] == pytest.approx(0.5329, abs=1e-6)
