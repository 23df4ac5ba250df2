"""Row f2 on the GPU (fstat_eval_batch_bands: per-template bands and segment limits) against
the oracle's `fstat_bands`, element by element through the C ABI.  Integer results (band limits) bit-exact;
F and F_k to north_star's 1e-5 relative."""
import numpy as np
import pytest

import synthetic as syn

pytestmark = pytest.mark.gpu

RTOL = 1e-5


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


@pytest.fixture(scope="module")
def bands(orc):
    return syn.make_dataset(syn.BANDS_SMALL, orc.template)


def _gpu(fs, ds, par, n_seg, lattice, opts=None):
    import torch
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(1), opts) as plan:
        p = torch.as_tensor(np.ascontiguousarray(par), device="cuda")
        F, Fk, band = fs.fstat_eval_batch_bands(plan, p, n_seg, lattice)
        torch.cuda.synchronize()
        return F.cpu().numpy(), Fk.cpu().numpy(), band.cpu().numpy()


def _check(orc, ds, par, n_seg, lattice, F, Fk, band):
    F_o, Fk_o, edges = orc.fstat_bands(ds.freq, ds.dw, ds.inv_sn, par, n_seg, lattice)
    T = ds.cfg.T
    for p in range(par.shape[0]):
        if orc.params_valid(par[p]):
            assert tuple(band[p]) == orc.template_band(par[p], ds.freq, T)
    live = np.isfinite(Fk_o) & (Fk_o != 0.0)
    assert np.array_equal(np.isneginf(Fk), np.isneginf(Fk_o))
    assert np.all(Fk[Fk_o == 0.0] == 0.0)                  # empty partitions and empty bands: exactly zero
    assert np.max(np.abs(Fk[live] - Fk_o[live]) / np.abs(Fk_o[live])) <= RTOL
    ok = np.isfinite(F_o) & (F_o != 0.0)
    assert np.array_equal(np.isneginf(F), np.isneginf(F_o)) and np.all(F[F_o == 0.0] == 0.0)
    assert np.max(np.abs(F[ok] - F_o[ok]) / np.abs(F_o[ok])) <= RTOL
    return int(live.sum())


@pytest.mark.parametrize("n_seg,lattice,full_model", [(1, 1, 0), (4, 1, 0), (16, 1, 0), (16, 64, 0), (64, 128, 0),
                                                       (7, 3, 0), (500, 1, 0), (4, 1, 1), (7, 3, 1), (64, 128, 1)])
def test_bands_small_every_F_and_Fk(fs, orc, bands, n_seg, lattice, full_model):
    """64 particles whose bands start below, inside and above the grid (39 non-empty), every F and F_k, through
    the three paths: lattice >= 32 (interpolating kernel over the lattice cells), lattice < 32 (the same over
    64-bin cells plus the pieces of the cells the edges split; 500 partitions put several edges into one cell),
    and force_level = -1 (full model at every in-band bin, per-thread edges)."""
    ds = bands
    par = syn.draw_particles(ds.cfg)
    opts = fs.fstat_default_options()
    opts.force_level = -1 if full_model else -2
    F, Fk, band = _gpu(fs, ds, par, n_seg, lattice, opts)
    n = _check(orc, ds, par, n_seg, lattice, F, Fk, band)
    assert n >= 30 * n_seg


@pytest.mark.parametrize("seg", [64, 320, 4096, 1 << 20])
def test_bands_work_segment_length_does_not_matter(fs, orc, bands, seg):
    """Work segments of one tile, a few tiles, many tiles, and one segment for the whole grid: partitions
    that lie inside one work segment, straddle two, or span many are all stitched the same."""
    ds = bands
    par = syn.draw_particles(ds.cfg)[:40]
    opts = fs.fstat_default_options()
    opts.max_segment_bins = seg
    opts.force_level = -1                                  # the kernel with per-thread edges (full model at every bin)
    F, Fk, band = _gpu(fs, ds, par, 16, 1, opts)
    _check(orc, ds, par, 16, 1, F, Fk, band)


def test_bands_invalid_particles_and_more_partitions_than_cells(fs, orc, bands):
    ds = bands
    par = syn.draw_particles(ds.cfg)[:12].copy()
    par[1, 1] = -3.0
    par[4, 2] = 0.3
    par[7, 0] = np.nan
    # 200 partitions on a 1024-bin lattice: bands of fewer than 200 cells leave empty partitions
    F, Fk, band = _gpu(fs, ds, par, 200, 1024)
    _check(orc, ds, par, 200, 1024, F, Fk, band)
    assert np.all(band[[1, 4, 7]] == 0)


def test_bands_repeatable_and_independent_of_batch_order(fs, bands):
    import torch
    ds = bands
    par = syn.draw_particles(ds.cfg)
    F1, Fk1, b1 = _gpu(fs, ds, par, 16, 1)
    F2, Fk2, b2 = _gpu(fs, ds, par, 16, 1)
    assert np.array_equal(F1, F2) and np.array_equal(Fk1, Fk2) and np.array_equal(b1, b2)
    perm = np.random.default_rng(0).permutation(par.shape[0])
    F3, Fk3, b3 = _gpu(fs, ds, par[perm], 16, 1)
    assert np.array_equal(F3, F1[perm]) and np.array_equal(Fk3, Fk1[perm]) and np.array_equal(b3, b1[perm])


@pytest.fixture(scope="module")
def first_stage(orc):
    return syn.make_dataset(syn.CONFIGS[1], orc.template)


@pytest.mark.parametrize("lattice", [1, 64])
def test_bands_host_buffers_give_the_same_bits(fs, bands, lattice):
    ds = bands
    par = syn.draw_particles(ds.cfg)
    F, Fk, band = _gpu(fs, ds, par, 16, lattice)
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(1)) as plan:
        F_h, Fk_h, band_h = fs.fstat_eval_batch_bands_host(plan, par, 16, lattice)
        import torch
        F_p, Fk_p, band_p = fs.fstat_eval_batch_bands_host(plan, torch.as_tensor(par).pin_memory(), 16, lattice)    # pinned tensors
    assert np.array_equal(F, F_h) and np.array_equal(Fk, Fk_h) and np.array_equal(band, band_h)
    assert F_p.is_pinned() and np.array_equal(F, F_p.numpy()) and np.array_equal(Fk, Fk_p.numpy()) and np.array_equal(band, band_p.numpy())


@pytest.mark.parametrize("lattice", [1, 64])
def test_bands_first_stage_sample(fs, orc, first_stage, lattice):
    """Config 1's data and particles (2.5 yr, 1 577 880 bins, N_seg = 1024) in the launch configuration
    bench.py --bands times (lattice 1: every in-band bin in full; lattice 64: the interpolating kernel over
    the lattice cells); a sample of particles against the oracle, every F_k of the sample."""
    import torch
    ds = first_stage
    par = syn.draw_particles(ds.cfg)
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(1)) as plan:
        p = torch.as_tensor(np.ascontiguousarray(par), device="cuda")
        F, Fk, band = fs.fstat_eval_batch_bands(plan, p, 1024, lattice)
        torch.cuda.synchronize()
        F, Fk, band = F.cpu().numpy(), Fk.cpu().numpy(), band.cpu().numpy()
    width = band[:, 1] - band[:, 0]
    assert (width > 0).sum() > 1500
    order = np.argsort(width)
    sample = np.unique(np.concatenate([order[-2:], order[(width[order] > 0).argmax():][:2], np.arange(0, 2048, 66)]))   # 35 particles
    _check(orc, ds, par[sample], 1024, lattice, F[sample], Fk[sample], band[sample])


@pytest.mark.parametrize("cfg_i,n_seg,lattice", [(1, 1024, 64), (2, 16, 128), (3, 1, 512), (1, 1024, 1), (2, 16, 1)])
def test_bands_interpolating_kernel_against_full_model_every_value(fs, orc, first_stage, cfg_i, n_seg, lattice):
    """At full size every F and F_k of the interpolating kernel over the lattice cells against the kernel that
    evaluates the full model at every in-band bin (force_level = -1; itself checked against the oracle above)
    with the same lattice.  5e-6 leaves the other half of north_star's 1e-5 to the full-model kernel."""
    import torch
    ds = first_stage                                      # configs 1-3 share the data; the particles differ
    par = syn.draw_particles(syn.CONFIGS[cfg_i])
    direct = fs.fstat_default_options()
    direct.force_level = -1
    out = []
    for opts in (None, direct):
        with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(1), opts) as plan:
            p = torch.as_tensor(np.ascontiguousarray(par), device="cuda")
            F, Fk, band = fs.fstat_eval_batch_bands(plan, p, n_seg, lattice)
            torch.cuda.synchronize()
            out.append((F.cpu().numpy(), Fk.cpu().numpy(), band.cpu().numpy()))
    (F_a, Fk_a, b_a), (F_b, Fk_b, b_b) = out
    assert np.array_equal(b_a, b_b)
    assert np.array_equal(Fk_a == 0.0, Fk_b == 0.0)
    live = Fk_b != 0.0
    assert live.sum() > 0.2 * live.size
    assert np.max(np.abs(Fk_a[live] - Fk_b[live]) / np.abs(Fk_b[live])) <= 5e-6
    ok = F_b != 0.0
    assert np.max(np.abs(F_a[ok] - F_b[ok]) / np.abs(F_b[ok])) <= 5e-6


def test_bands_wide_band_in_particle_batches(fs, orc):
    """Config 4's grid (7.1 M bins to 100 mHz, across the TDI null): 111 k lattice cells make the record
    workspace 8.9 MB per particle, so P = 4096 is evaluated in two particle batches.  A sample against the oracle,
    and the whole batch against the same particles evaluated 512 at a time (other groups, other strides)."""
    import torch
    cfg = syn.CONFIGS[4]
    ds = syn.make_dataset(cfg, orc.template)
    par = syn.draw_particles(cfg, 4096)
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(1)) as plan:
        p = torch.as_tensor(np.ascontiguousarray(par), device="cuda")
        F, Fk, band = fs.fstat_eval_batch_bands(plan, p, 16, 64)
        torch.cuda.synchronize()
        parts = [fs.fstat_eval_batch_bands(plan, p[i:i + 512].contiguous(), 16, 64) for i in range(0, 4096, 512)]
        torch.cuda.synchronize()
    F, Fk, band = F.cpu().numpy(), Fk.cpu().numpy(), band.cpu().numpy()
    F2 = np.concatenate([q[0].cpu().numpy() for q in parts])
    Fk2 = np.concatenate([q[1].cpu().numpy() for q in parts])
    b2 = np.concatenate([q[2].cpu().numpy() for q in parts])
    assert np.array_equal(band, b2) and np.array_equal(Fk == 0.0, Fk2 == 0.0)
    live = Fk2 != 0.0
    assert live.sum() > 0.5 * live.size
    assert np.max(np.abs(Fk[live] - Fk2[live]) / np.abs(Fk2[live])) <= 5e-6
    sample = np.array([0, 1500, 2047, 2048, 3000, 4095])      # both batches
    _check(orc, ds, par[sample], 16, 64, F[sample], Fk[sample], band[sample])


@pytest.mark.parametrize("lattice", [1, 64])
def test_bands_odd_sizes(fs, orc, lattice):
    """A grid whose length is 3 modulo 64 (the last cell is shorter than the smallest node stride and goes to the
    direct kernel), 37 particles (a partly filled group), 5 partitions."""
    import dataclasses
    T = syn.BANDS_SMALL.T
    cfg = dataclasses.replace(syn.BANDS_SMALL, f_lo=0.020, f_hi=(380348 + 0.5) / T)
    ds = syn.make_dataset(cfg, orc.template)
    assert ds.n_bins % 64 == 3
    par = syn.draw_particles(cfg, 37)
    par[:, 0] = np.linspace(0.9, 2.2, 37) * syn.YEAR_S       # several bands reach the end of the grid
    F, Fk, band = _gpu(fs, ds, par, 5, lattice)
    n = _check(orc, ds, par, 5, lattice, F, Fk, band)
    assert n >= 30 and (band[:, 1] == ds.n_bins).sum() >= 3


@pytest.mark.parametrize("n_seg", [256, 1024])
def test_bands_narrow_bands_and_short_partitions_against_full_model(fs, n_seg):
    """A harder population than BASELINE.json's (M_c 10-60, e_0 up to 0.3) on the 2.5-yr grid: slowly evolving
    templates have bands of a few thousand bins, i.e. partitions far shorter than a cell.  A partition with no whole
    cell inside is evaluated edge to edge with the full model (an earlier version built it from differences of cell
    records and was off by up to 7e-4 there: short partitions have a near-singular M_k and amplify the interpolation
    error of a record); every F_k of partitions of >= 16 bins against the full-model kernel.  (Shorter ones are
    beyond FP64 for any evaluation order.)"""
    import torch
    from synthetic import lisa_data as L
    cfg = syn.CONFIGS[1]
    _, n, f = syn.frequency_grid(cfg.T, cfg.f_lo, cfg.f_hi)
    sn = syn.psd_tdi_x(f)
    d = syn.coloured_noise(sn, cfg.T, 7)
    rng = np.random.default_rng(1003)
    par = L._wide_particles(rng, 2048, cfg.T)
    par[:, 5] = rng.uniform(0.0, 0.3, 2048)
    par[:, 1] = rng.uniform(10.0, 60.0, 2048)
    direct = fs.fstat_default_options()
    direct.force_level = -1
    out = []
    for opts in (None, direct):
        with fs.fstat_plan_create(f, d / sn, 1.0 / sn, syn.equal_bin_edges(n, 1), opts) as plan:
            p = torch.as_tensor(par, device="cuda")
            F, Fk, band = fs.fstat_eval_batch_bands(plan, p, n_seg, 1)
            torch.cuda.synchronize()
            out.append((Fk.cpu().numpy(), band.cpu().numpy()))
    (Fk_a, b_a), (Fk_b, b_b) = out
    assert np.array_equal(b_a, b_b) and np.array_equal(Fk_a == 0.0, Fk_b == 0.0)
    width = b_a[:, 1] - b_a[:, 0]
    assert ((width > 0) & (width < 64 * n_seg)).sum() >= 10          # templates whose partitions are shorter than a cell
    long_enough = (width // n_seg >= 16)[:, None] & (Fk_b != 0.0)
    assert np.max(np.abs(Fk_a[long_enough] - Fk_b[long_enough]) / np.abs(Fk_b[long_enough])) <= 5e-6
