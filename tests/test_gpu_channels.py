"""Row f4 on the GPU (fstat_eval_batch_channels: the channel sum of PAPER.md:62 Eq. 3) against the oracle's
`fstat_batch_channels`, element by element through the C ABI; 1e-5 relative on every F and F_k."""
import dataclasses
import math

import numpy as np
import pytest

import synthetic as syn

pytestmark = pytest.mark.gpu

RTOL = 1e-5
LAM = 2.0 * math.pi / 3.0


@pytest.fixture(scope="module")
def fs():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2407_10797_b200 import build
    build.build()
    import paper_2407_10797_b200 as fs
    fs.load_library()
    return fs


def _channels(orc, cfg, n):
    """n data sets of one config: channel c sees the response with orbit_lambda = 2 pi c / 3 (X, Y, Z), its own noise
    seed and the injection through its own response."""
    out = []
    for c in range(n):
        o = orc.default_options(orbit_lambda=c * LAM)
        ds = syn.make_dataset(dataclasses.replace(cfg, noise_seed=50 + c), lambda p, f, o=o: orc.template(p, f, o))
        out.append((ds, o))
    return out


def _gpu(fs, chans, edges, par, **opt_kw):
    import torch
    plans = []
    try:
        for c, (ds, _) in enumerate(chans):
            o = fs.fstat_default_options()
            o.orbit_lambda = c * LAM
            for k, v in opt_kw.items():
                setattr(o, k, v)
            plans.append(fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges, o))
        p = torch.as_tensor(np.ascontiguousarray(par), device="cuda")
        F, Fk = fs.fstat_eval_batch_channels(plans, p)
        torch.cuda.synchronize()
        return F.cpu().numpy(), Fk.cpu().numpy()
    finally:
        for pl in plans:
            fs.fstat_plan_destroy(pl)


def _compare(orc, chans, edges, par, F, Fk):
    ds0 = chans[0][0]
    F_o, Fk_o = orc.fstat_batch_channels(ds0.freq, [(ds.dw, ds.inv_sn, o) for ds, o in chans], edges, par)
    fin = np.isfinite(Fk_o)
    assert np.array_equal(np.isneginf(Fk), ~fin)
    assert np.max(np.abs(Fk[fin] - Fk_o[fin]) / np.abs(Fk_o[fin])) <= RTOL
    ok = np.isfinite(F_o)
    assert np.array_equal(np.isneginf(F), ~ok)
    assert np.max(np.abs(F[ok] - F_o[ok]) / np.abs(F_o[ok])) <= RTOL


@pytest.mark.parametrize("n_ch", [1, 2, 3])
def test_tiny_channels_every_F_and_Fk(fs, orc, n_ch):
    cfg = syn.CONFIGS[0]
    chans = _channels(orc, cfg, n_ch)
    par = syn.draw_particles(cfg).copy()
    par[5, 1] = -1.0                                       # one invalid particle flies
    edges = chans[0][0].edges(4)
    F, Fk = _gpu(fs, chans, edges, par)
    _compare(orc, chans, edges, par, F, Fk)


def test_fine_slice_three_channels_through_the_interpolating_kernel(fs, orc):
    """A 2.5-yr slice (the interpolating kernel does all the work), X + Y + Z, every F and F_k."""
    year = syn.YEAR_S
    cfg = syn.Config(17, "ch_slice", 2.5 * year, 0.0200, 0.0202, (8,), (96,), 3.5 * year, "wide")
    chans = _channels(orc, cfg, 3)
    par = syn.draw_particles(cfg)
    edges = chans[0][0].edges(8)
    F, Fk = _gpu(fs, chans, edges, par)
    _compare(orc, chans, edges, par, F, Fk)
    F_d, Fk_d = _gpu(fs, chans, edges, par, force_level=-1)          # the direct kernel gives the same
    assert np.max(np.abs(Fk - Fk_d) / np.abs(Fk_d)) <= 5e-6


def test_first_stage_two_channels_sample(fs, orc):
    """Config 1 at full size (N_p = 1024, P = 2048) with two channels; a sample of particles against the oracle."""
    cfg = syn.CONFIGS[1]
    chans = _channels(orc, cfg, 2)
    par = syn.draw_particles(cfg)
    edges = chans[0][0].edges(1024)
    F, Fk = _gpu(fs, chans, edges, par)
    sample = np.array([0, 167, 511, 1024, 1598, 2047])
    _compare(orc, chans, edges, par[sample], F[sample], Fk[sample])


# ------------------------------------------------------------------------------------------ A, E, T (reading A28)
def _aet_channels(orc, cfg, names, snr=None):
    """One data set per TDI combination: its own noise PSD (synthetic.psd_tdi), noise seed, and the injection seen
    through its own response (the oracle's template with tdi_channel set)."""
    out = []
    for c, name in enumerate(names):
        o = orc.default_options(tdi_channel=orc.TDI_CHANNELS[name])
        ds = syn.make_dataset(dataclasses.replace(cfg, noise_seed=70 + c), lambda p, f, o=o: orc.template(p, f, o),
                              channel=name, snr=snr)
        out.append((ds, o, name))
    return out


def _gpu_named(fs, chans, edges, par, **opt_kw):
    import torch
    plans = []
    try:
        for ds, _, name in chans:
            o = fs.fstat_default_options(tdi_channel=fs.TDI_CHANNELS[name], **opt_kw)
            plans.append(fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges, o))
        p = torch.as_tensor(np.ascontiguousarray(par), device="cuda")
        F, Fk = fs.fstat_eval_batch_channels(plans, p)
        torch.cuda.synchronize()
        return F.cpu().numpy(), Fk.cpu().numpy()
    finally:
        for pl in plans:
            fs.fstat_plan_destroy(pl)


@pytest.mark.parametrize("names", ["Y", "Z", "A", "E", "T", "AET", "XYZ"])
def test_tiny_every_channel_and_the_aet_sum_every_F_and_Fk(fs, orc, names):
    """Every TDI combination the library templates, alone and (A, E, T: the set with independent noise)
    summed as in Eq. 3, on config 0 through the direct kernel: every F and F_k against the oracle."""
    cfg = syn.CONFIGS[0]
    chans = _aet_channels(orc, cfg, names)
    par = syn.draw_particles(cfg).copy()
    par[9, 2] = 0.3                                        # one invalid particle flies
    edges = chans[0][0].edges(4)
    F, Fk = _gpu_named(fs, chans, edges, par)
    _compare(orc, [(ds, o) for ds, o, _ in chans], edges, par, F, Fk)


def test_aet_templates_match_the_oracle_bin_by_bin(fs, orc):
    import torch
    cfg = syn.CONFIGS[0]
    ds = syn.make_dataset(cfg, None)
    par = syn.draw_particles(cfg)
    for name in "YZAET":
        with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(1),
                                  fs.fstat_default_options(tdi_channel=fs.TDI_CHANNELS[name])) as plan:
            for p in (3, 40):
                up_o, uc_o = orc.template(par[p], ds.freq, orc.default_options(tdi_channel=orc.TDI_CHANNELS[name]))
                up_g, uc_g = fs.fstat_eval_template(plan, par[p])
                scale = max(np.abs(up_o).max(), np.abs(uc_o).max())
                assert np.abs(up_g.cpu().numpy() - up_o).max() <= 1e-7 * scale, name
                assert np.abs(uc_g.cpu().numpy() - uc_o).max() <= 1e-7 * scale, name


def test_fine_slice_aet_through_the_interpolating_kernel(fs, orc):
    """A 2.5-yr slice, A + E + T, every F and F_k: the interpolating kernel with the A / E / T response at its nodes
    against the oracle, and against the direct kernel."""
    year = syn.YEAR_S
    cfg = syn.Config(18, "aet_slice", 2.5 * year, 0.0200, 0.0202, (8,), (96,), 3.5 * year, "wide")
    chans = _aet_channels(orc, cfg, "AET")
    par = syn.draw_particles(cfg)
    edges = chans[0][0].edges(8)
    F, Fk = _gpu_named(fs, chans, edges, par)
    _compare(orc, [(ds, o) for ds, o, _ in chans], edges, par, F, Fk)
    F_d, Fk_d = _gpu_named(fs, chans, edges, par, force_level=-1)
    assert np.max(np.abs(Fk - Fk_d) / np.abs(Fk_d)) <= 5e-6


@pytest.mark.parametrize("names", ["AET", "AE", "TA"])
def test_fused_pass_equals_one_pass_per_channel(fs, orc, names):
    """Two or three A / E / T plans go through one pass of the fused interpolating kernel (csrc/fstat_fastmulti.cu);
    options.no_channel_fusion sends the same plans through one pass per channel.  The two share the node model, the
    carrier recurrence and the order of every sum, so they agree to rounding; ragged partition edges cut node intervals
    and the fused kernel's 256-bin tiles at arbitrary bins, and a wide-stride level is forced so that a 512-bin
    interval spans two tiles."""
    year = syn.YEAR_S
    cfg = syn.Config(19, "aet_fused", 2.5 * year, 0.0200, 0.0203, (8,), (200,), 3.5 * year, "wide")
    chans = _aet_channels(orc, cfg, names)
    par = syn.draw_particles(cfg)
    n = chans[0][0].freq.size
    edges = np.array([0, 1001, 2750, 2763, 5000, 7777, 9013, n - 5, n], dtype=np.int64)
    for kw in ({}, {"force_level": 6}, {"force_level": 0}):
        F_f, Fk_f = _gpu_named(fs, chans, edges, par, **kw)
        F_s, Fk_s = _gpu_named(fs, chans, edges, par, no_channel_fusion=1, **kw)
        assert np.max(np.abs(Fk_f - Fk_s) / np.abs(Fk_s)) <= 1e-10, kw
        assert np.max(np.abs(F_f - F_s) / np.abs(F_s)) <= 1e-10, kw
    F, Fk = _gpu_named(fs, chans, edges, par)
    _compare(orc, [(ds, o) for ds, o, _ in chans], edges, par, F, Fk)


def test_first_stage_aet_sample(fs, orc):
    """Config 1 at full size (N_p = 1024, P = 2048) with A + E + T; 64 particles against the oracle (through
    the fused three-channel kernel)."""
    cfg = syn.CONFIGS[1]
    chans = _aet_channels(orc, cfg, "AET")
    par = syn.draw_particles(cfg)
    edges = chans[0][0].edges(1024)
    F, Fk = _gpu_named(fs, chans, edges, par)
    sample = np.arange(5, 2048, 32)                        # 64 particles, every F_k of each
    _compare(orc, [(ds, o) for ds, o, _ in chans], edges, par[sample], F[sample], Fk[sample])


def test_bands_refuse_aet_plans(fs, orc):
    import torch
    cfg = syn.CONFIGS[0]
    ds = syn.make_dataset(cfg, None)
    par = torch.as_tensor(syn.draw_particles(cfg), device="cuda")
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(1), fs.fstat_default_options(tdi_channel=3)) as plan:
        with pytest.raises(fs.FstatError) as ei:
            fs.fstat_eval_batch_bands(plan, par, 4, 1)
        assert ei.value.status == 4


def test_mismatching_plans_are_rejected(fs, orc):
    import torch
    cfg = syn.CONFIGS[0]
    ds = syn.make_dataset(cfg, orc.template)
    par = torch.as_tensor(syn.draw_particles(cfg), device="cuda")
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(4)) as a, \
         fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(2)) as b:
        with pytest.raises(fs.FstatError):
            fs.fstat_eval_batch_channels([a, b], par)
        with pytest.raises(fs.FstatError):
            fs.fstat_eval_batch_channels([a, a], par)
        F1, Fk1 = fs.fstat_eval_batch_channels([a], par)
        F0, Fk0 = fs.fstat_eval_batch(a, par)
        torch.cuda.synchronize()
        assert torch.equal(F1, F0) and torch.equal(Fk1, Fk0)       # one channel: the same kernels, the same bits
