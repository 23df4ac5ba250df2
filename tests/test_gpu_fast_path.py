"""The interpolating main kernel (fstat_fast.cu) against the CPU oracle, element by element, at sizes the
oracle finishes in seconds: a fine-grid (df = 1 / 2.5 yr) slice of the paper's band so that the stride
criterion admits every stride, ragged partitions that cut node intervals and data tiles, forced strides,
and the stride selection itself.  Bar: 1e-5 relative on every F and F_k (north_star).  ``-m gpu``."""
import numpy as np
import pytest

import synthetic as syn

pytestmark = pytest.mark.gpu

RTOL = 1e-5
YEAR = 31557600.0
T25 = 2.5 * YEAR


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
def torch_():
    import torch
    return torch


def _fine_cfg(f_lo, f_hi, index=9):
    return syn.Config(index, "fine_slice", T25, f_lo, f_hi, (8,), (48,), 3.5 * YEAR, "wide")


@pytest.fixture(scope="module")
def fine(orc):
    """7889 bins at 20 mHz on the 2.5-yr grid: noise (seed 0) + an SNR-12 injection from the oracle."""
    return syn.make_dataset(_fine_cfg(0.0200, 0.0201), orc.template)


def _rel(a, b):
    return np.abs(np.asarray(a) - np.asarray(b)) / np.abs(np.asarray(b))


def _eval(fs, torch, ds, edges, par, **opt):
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges, fs.fstat_default_options(**opt)) as plan:
        F, Fk = fs.fstat_eval_batch(plan, torch.as_tensor(np.ascontiguousarray(par), device="cuda"))
        torch.cuda.synchronize()
        bins, sub = fs.fstat_plan_level_bins(plan)
        return F.cpu().numpy(), Fk.cpu().numpy(), bins, sub


def test_auto_stride_matches_oracle_and_uses_the_interpolating_kernel(fs, torch_, orc, fine):
    ds = fine
    par = syn.draw_particles(ds.cfg, 48)
    edges = ds.edges(8)
    F_o, Fk_o = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par)
    F_g, Fk_g, bins, sub = _eval(fs, torch_, ds, edges, par)
    assert bins[0] == 0 and bins[1:].sum() == ds.n_bins          # one group of 128: every bin interpolated
    assert _rel(Fk_g, Fk_o).max() <= RTOL
    assert _rel(F_g, F_o).max() <= RTOL
    assert _rel(Fk_g, Fk_o).max() <= 2e-6                          # well inside the bar at the default tolerance


@pytest.mark.parametrize("level", [-1, 0, 1, 2, 3, 4, 5])
def test_every_forced_stride_matches_oracle(fs, torch_, orc, fine, level):
    """At 20 mHz every stride up to 256 bins is accurate for M_c >= 20 (orbital phase advance per bin
    ~5e-5 rad); -1 is the direct kernel."""
    ds = fine
    par = syn.draw_particles(ds.cfg, 40)
    edges = ds.edges(8)
    F_o, Fk_o = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par)
    F_g, Fk_g, bins, sub = _eval(fs, torch_, ds, edges, par, force_level=level)
    assert bins[level + 1] == ds.n_bins
    assert _rel(Fk_g, Fk_o).max() <= RTOL, level
    assert _rel(F_g, F_o).max() <= RTOL, level


def test_largest_stride_at_28_mhz(fs, torch_, orc):
    """Stride 512 (the largest) needs an orbital phase advance below ~2e-5 rad per bin: forced on a 28 mHz
    slice, where the automatic selection also picks it for most of the band."""
    ds = syn.make_dataset(_fine_cfg(0.0280, 0.0281, index=13), orc.template)
    par = syn.draw_particles(ds.cfg, 40)
    edges = ds.edges(2)
    F_o, Fk_o = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par)
    F_g, Fk_g, bins, _ = _eval(fs, torch_, ds, edges, par, force_level=6)
    assert bins[7] == ds.n_bins
    assert _rel(Fk_g, Fk_o).max() <= RTOL and _rel(F_g, F_o).max() <= RTOL
    par[:, 1] = np.linspace(32.0, 40.0, 40)
    edges = ds.edges(1)                                   # a wide partition: little near-singular amplification
    F_o, Fk_o = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par)
    F_g, Fk_g, bins, _ = _eval(fs, torch_, ds, edges, par)
    assert bins[7] > 0 and bins[0] == 0
    assert _rel(Fk_g, Fk_o).max() <= 2e-6 and _rel(F_g, F_o).max() <= 2e-6


def test_ragged_edges_cut_node_intervals_and_tiles(fs, torch_, orc, fine):
    """Partition edges that are not multiples of any stride, one-bin partitions (direct kernel: shorter
    than 8 bins; exactly singular M_k), partitions inside one node interval, and a partition spanning
    many 512-bin tiles; also through fstat_plan_set_partitions and with segment cuts every 512 / 1024
    bins.  (Partitions of 2-20 bins are left out on this fine grid: the template barely changes over
    them, M_k is singular to ~1e-12 and no FP64 evaluation, the oracle's included, is good to 1e-5.)"""
    ds = fine
    n = ds.n_bins
    par = syn.draw_particles(ds.cfg, 33)
    edge_sets = [
        np.array([0, 1, 25, 48, 300, 301, 767, 768, 1024, 1061, 2500, 2563, 7000, n]),
        np.array([0, 255, 256, 257, 511, 540, n - 40, n - 1, n]),
        np.array([0, n]),
        np.array([0, 100, 200, 250, 1000, 4096, n]),
    ]
    for seg in (0, 512, 1024):
        for level in (-2, 0, 5):
            opts = fs.fstat_default_options(max_segment_bins=seg, force_level=level)
            with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(1), opts) as plan:
                p = torch_.as_tensor(par, device="cuda")
                for edges in edge_sets:
                    edges = np.asarray(edges, dtype=np.int64)
                    fs.fstat_plan_set_partitions(plan, edges)
                    F_g, Fk_g = fs.fstat_eval_batch(plan, p)
                    torch_.cuda.synchronize()
                    bins, _ = fs.fstat_plan_level_bins(plan)
                    F_o, Fk_o = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par)
                    short = int(sum(b - a for a, b in zip(edges[:-1], edges[1:]) if b - a < 8)) if seg == 0 else None
                    if short is not None:
                        assert bins[0] == short          # only partitions shorter than 8 bins go direct
                    assert _rel(Fk_g.cpu().numpy(), Fk_o).max() <= RTOL, (seg, level, len(edges))
                    assert _rel(F_g.cpu().numpy(), F_o).max() <= RTOL, (seg, level, len(edges))


def test_low_frequency_slice_needs_small_strides(fs, torch_, orc):
    """At 10 mHz the orbital phase at t_f moves ~6e-4 rad per bin for M_c = 20: the criterion must pick
    small strides there (never 256) and still meet the bar; forcing stride 256 must NOT (which shows the
    criterion is doing real work)."""
    ds = syn.make_dataset(_fine_cfg(0.0100, 0.0101, index=10), None)
    par = syn.draw_particles(ds.cfg, 40)
    par[:, 1] = np.linspace(20.0, 24.0, 40)                       # low chirp masses: fastest t_f sweep
    edges = ds.edges(4)
    F_o, Fk_o = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par)
    F_g, Fk_g, bins, _ = _eval(fs, torch_, ds, edges, par)
    assert bins[4:].sum() == 0 and bins[:4].sum() == ds.n_bins     # nothing at stride >= 64
    assert _rel(Fk_g, Fk_o).max() <= RTOL and _rel(F_g, F_o).max() <= RTOL
    F_b, Fk_b, _, _ = _eval(fs, torch_, ds, edges, par, force_level=6)
    assert _rel(Fk_b, Fk_o).max() > 10 * _rel(Fk_g, Fk_o).max()


def test_tiny_config_runs_entirely_in_the_direct_kernel(fs, torch_, tiny):
    """Config 0 (T = 2^20 s) moves t_f by ~1e5 s per bin: no stride is admissible (hazard H7)."""
    ds = tiny
    par = syn.draw_particles(ds.cfg)
    _, _, bins, sub = _eval(fs, torch_, ds, ds.edges(4), par)
    assert bins[0] == ds.n_bins and bins[1:].sum() == 0 and sub.sum() == 0


def test_tolerance_option_moves_the_strides(fs, torch_, orc):
    ds = syn.make_dataset(_fine_cfg(0.0130, 0.0131, index=11), None)
    par = syn.draw_particles(ds.cfg, 16)
    edges = ds.edges(2)
    _, _, b1, _ = _eval(fs, torch_, ds, edges, par)
    _, _, b2, _ = _eval(fs, torch_, ds, edges, par, interp_tol=1e-3)
    _, _, b3, _ = _eval(fs, torch_, ds, edges, par, interp_tol=1e3)
    mean = lambda b: float((b[1:] * (8 << np.arange(7))).sum()) / max(int(b[1:].sum()), 1)
    assert mean(b2) < mean(b1) < mean(b3)
    with pytest.raises(fs.FstatError):
        fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges, fs.fstat_default_options(interp_tol=0.0))
    with pytest.raises(fs.FstatError):
        fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges, fs.fstat_default_options(force_level=7))


def test_grid_starting_near_zero_frequency_falls_back_to_direct(fs, torch_, orc):
    """The node grid reaches 512 bins below the band; a band that starts closer to f = 0 than that cannot
    be interpolated and must run (correctly) in the direct kernel."""
    T = T25
    k = np.arange(100, 400)
    f = k / T * 1e4                                              # 12.7 uHz .. : coarse grid near zero
    rng = np.random.default_rng(3)
    sn = np.ones(f.size)
    d = rng.standard_normal(f.size) + 1j * rng.standard_normal(f.size)
    par = syn.draw_particles(syn.CONFIGS[1], 4)

    class DS:
        freq, dw, inv_sn = f, d / sn, 1.0 / sn
        n_bins = f.size
    edges = np.array([0, 150, f.size])
    F_o, Fk_o = orc.fstat_batch(f, DS.dw, DS.inv_sn, edges, par)
    F_g, Fk_g, bins, _ = _eval(fs, torch_, DS, edges, par, force_level=2)
    assert bins[0] == f.size
    assert _rel(Fk_g, Fk_o).max() <= RTOL


def _source_along_arm(orc, arm, sign, tc, f_mid):
    """Parameters of a source whose propagation direction is (anti)parallel to arm 1 -> arm+1 at t_f(f_mid):
    there k.n = +-|n| with n = (p_j - p_1)/L NOT of unit length (reading A10), so 1 - |k.n| changes sign."""
    base = np.array([tc, 30.0, 0.24, 1.0, 1.0, 0.03])
    _, tf = orc.phase(base, f_mid)                       # t_f does not depend on the sky position
    p = orc.orbit(tf)
    n = (p[arm] - p[0]) / 2.5e9
    src = -sign * n / np.linalg.norm(n)                   # k = -(direction to the source)
    base[3] = float(np.arccos(src[2]))
    base[4] = float(np.arctan2(src[1], src[0]) % (2.0 * np.pi))
    return base, float(np.linalg.norm(n))


def test_source_along_a_breathing_arm(fs, torch_, orc, fine):
    """|k.n| crosses 1 when the source lies along an arm that is longer than nominal: the sinc arguments
    x (1 -+ k.n) change sign there.  Direct and interpolating kernels against the oracle."""
    ds = fine
    f_mid = float(ds.freq[ds.n_bins // 2])
    par, norms = [], []
    for arm in (1, 2):
        for sign in (1.0, -1.0):
            for tc in (3.1 * YEAR, 3.5 * YEAR, 3.9 * YEAR, 4.4 * YEAR):
                q, nn = _source_along_arm(orc, arm, sign, tc, f_mid)
                par.append(q)
                norms.append(nn)
    par = np.array(par)
    assert max(norms) > 1.001 and min(norms) < 0.999     # both signs of 1 - |n| are exercised
    edges = ds.edges(8)
    F_o, Fk_o = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par)
    for level in (-1, -2):
        F_g, Fk_g, _, _ = _eval(fs, torch_, ds, edges, par, force_level=level)
        assert _rel(Fk_g, Fk_o).max() <= RTOL, level
        assert _rel(F_g, F_o).max() <= RTOL, level
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges) as plan:
        for i in (0, 5, 10, 15):
            up_o, uc_o = orc.template(par[i], ds.freq)
            up_g, uc_g = fs.fstat_eval_template(plan, par[i])
            scale = max(np.abs(up_o).max(), np.abs(uc_o).max())
            assert np.abs(up_g.cpu().numpy() - up_o).max() <= 1e-7 * scale
            assert np.abs(uc_g.cpu().numpy() - uc_o).max() <= 1e-7 * scale
