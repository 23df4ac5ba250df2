"""PSO on the device.  CPU: the oracle's generator against the Random123 known answers, its
update rule against closed-form cases.  GPU: the device swarm state against the oracle step by step (bit for
bit in x and v when the oracle is fed the device's fitness values), let-them-fly, batched swarms."""
import json
import os

import numpy as np
import pytest

import synthetic as syn
from oracle import pso_oracle as po

HERE = os.path.dirname(os.path.abspath(__file__))


def test_philox_matches_the_random123_known_answers():
    kat = json.load(open(os.path.join(HERE, "golden", "philox4x32_10_kat.json")))
    for v in kat["vectors"]:
        c = [int(x, 16) for x in v["counter"]]
        k = [int(x, 16) for x in v["key"]]
        out = po.philox4x32_10(*[np.array([x], dtype=np.uint64) for x in c], k[0], k[1])
        assert ["%08x" % int(o[0]) for o in out] == v["output"]


def test_uniforms_are_uniform_and_counter_based():
    u = po.uniforms12(20000, 3, 12345)
    assert u.min() > 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.005 and abs(u.var() - 1.0 / 12.0) < 0.002
    np.testing.assert_array_equal(po.uniforms12(100, 3, 12345), u[:100])          # no hidden state
    assert not np.array_equal(po.uniforms12(100, 4, 12345), u[:100])
    assert not np.array_equal(po.uniforms12(100, 3, 12346), u[:100])


def test_oracle_update_rule_closed_forms():
    x, v = po.init(2, 5, seed=9)
    assert x.shape == (10, 6) and np.all(np.abs(v) <= 0.5) and np.all((x > 0) & (x < 1))
    pbest, pbest_f = x.copy(), np.arange(10, dtype=float)
    # c1 = c2 = 0: pure inertia, w = w_start at the first iteration
    x1, v1 = po.step(x, v, pbest, pbest_f, 5, 1, 10, 9, c1=0.0, c2=0.0, v_max=10.0)
    np.testing.assert_allclose(v1, 0.9 * v, rtol=0, atol=1e-16)
    np.testing.assert_allclose(x1, x + 0.9 * v, rtol=0, atol=1e-16)
    assert po.inertia(10, 10) == pytest.approx(0.4) and po.inertia(1, 10) == 0.9
    # zero velocity, pbest = x, c1 = 0: the particle moves only towards its ring-best neighbour
    x2, v2 = po.step(x, np.zeros_like(v), pbest, pbest_f, 5, 1, 10, 9, c1=0.0, c2=2.0, v_max=10.0)
    u = po.uniforms12(10, 1, 9)
    # particle 0 of swarm 0: neighbours 4, 0, 1 with fitness 4, 0, 1 -> lbest = particle 4
    np.testing.assert_allclose(v2[0], 2.0 * u[0, 6:] * (x[4] - x[0]), rtol=1e-15)
    # particle 2 of swarm 1 (gid 7): neighbours 6, 7, 8 -> lbest = 8
    np.testing.assert_allclose(v2[7], 2.0 * u[7, 6:] * (x[8] - x[7]), rtol=1e-15)
    # out of the box -> NaN parameters; better fitness replaces the personal best, equal does not
    par = po.to_params(np.array([[0.5] * 6, [0.5, 1.2, 0.5, 0.5, 0.5, 0.5]]), np.zeros(6), np.full(6, 2.0))
    assert np.all(par[0] == 1.0) and np.all(np.isnan(par[1]))
    pb, pf = po.update_best(x1, np.array([0.0, 5.0] * 5), pbest, pbest_f)
    assert np.array_equal(pb[1], x1[1]) and np.array_equal(pb[0], pbest[0]) and pf[1] == 5.0 and pf[0] == 0.0


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2407_10797_b200 import build
    build.build()
    import paper_2407_10797_b200 as fs
    fs.load_library()
    return fs


@pytest.mark.gpu
def test_device_swarms_follow_the_oracle_step_by_step(gpu, orc):
    fs = gpu
    year = 31557600.0
    cfg = syn.Config(15, "pso_slice", 2.5 * year, 0.0200, 0.0201, (4,), (64,), 3.5 * year, "wide")
    ds = syn.make_dataset(cfg, orc.template)
    inj = ds.inj_params
    lo = np.array([inj[0] - 3000.0, inj[1] * 0.998, 0.2, inj[3] - 0.1, inj[4] - 0.1, 0.0])
    hi = np.array([inj[0] + 3000.0, inj[1] * 1.002, 0.25, inj[3] + 0.1, inj[4] + 0.1, 0.1])
    n_swarms, n_part, n_iter, seed = 3, 24, 12, 0x1234567890ABCDEF
    edges = ds.edges(4)
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges) as plan:
        with fs.fstat_pso_create(plan, n_swarms, n_part, n_iter, lo, hi, seed) as pso:
            x_o, v_o = po.init(n_swarms, n_part, seed)
            x, v, pb, pf, fl = fs.fstat_pso_state(pso)
            np.testing.assert_array_equal(x, x_o)                  # bit for bit
            np.testing.assert_array_equal(v, v_o)
            np.testing.assert_array_equal(pb, x_o)
            np.testing.assert_array_equal(pf, fl)
            F_o, _ = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, po.to_params(x_o, lo, hi))
            assert np.max(np.abs(fl - F_o) / np.abs(F_o)) <= 1e-5  # the fitness is the oracle's F
            pb_o, pf_o = x_o.copy(), fl.copy()                     # from here on the oracle is fed the device's F
            seen_outside = 0
            for it in range(1, n_iter + 1):
                fs.fstat_pso_iterate(pso, 1)
                x, v, pb, pf, fl = fs.fstat_pso_state(pso)
                x_o, v_o = po.step(x_o, v_o, pb_o, pf_o, n_part, it, n_iter, seed)
                np.testing.assert_array_equal(x, x_o, err_msg="iteration %d" % it)
                np.testing.assert_array_equal(v, v_o)
                par_o = po.to_params(x_o, lo, hi)
                outside = np.isnan(par_o[:, 0])
                seen_outside += int(outside.sum())
                assert np.all(np.isneginf(fl[outside])) and np.all(np.isfinite(fl[~outside]))
                pb_o, pf_o = po.update_best(x_o, fl, pb_o, pf_o)
                np.testing.assert_array_equal(pb, pb_o)
                np.testing.assert_array_equal(pf, pf_o)
                if it in (1, n_iter):                                # spot-check the fitness against the oracle
                    F_o, _ = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par_o[~outside])
                    assert np.max(np.abs(fl[~outside] - F_o) / np.abs(F_o)) <= 1e-5
            assert fs.fstat_pso_iterations_done(pso) == n_iter and seen_outside > 0      # some did fly out
            bp, bf = fs.fstat_pso_best(pso)
            for s in range(n_swarms):
                sl = slice(s * n_part, (s + 1) * n_part)
                j = int(np.argmax(pf_o[sl]))
                assert bf[s] == pf_o[sl][j]
                np.testing.assert_allclose(bp[s], lo + pb_o[sl][j] * (hi - lo), rtol=0, atol=0)


@pytest.mark.gpu
def test_one_box_per_swarm(gpu, orc):
    """fstat_pso_create_boxes: three swarms, three different boxes (the hierarchy's stages search one box per t_c
    interval / candidate).  The unit-box state is the oracle's (which never sees the boxes), the
    physical parameters follow each swarm's own box bit for bit, and every best lies inside its swarm's box."""
    fs = gpu
    cfg = syn.CONFIGS[0]
    ds = syn.make_dataset(cfg, orc.template)
    inj = ds.inj_params
    n_swarms, n_part, n_iter, seed = 3, 16, 4, 99
    lo = np.array([[inj[0] - 3000.0 * (s + 1), inj[1] * (0.998 - 0.001 * s), 0.2, inj[3] - 0.1, inj[4] - 0.1, 0.0] for s in range(3)])
    hi = np.array([[inj[0] + 3000.0 * (s + 1), inj[1] * (1.002 + 0.001 * s), 0.25, inj[3] + 0.1, inj[4] + 0.1, 0.1] for s in range(3)])
    edges = ds.edges(4)
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges) as plan:
        with fs.fstat_pso_create(plan, n_swarms, n_part, n_iter, lo, hi, seed) as pso:
            x_o, v_o = po.init(n_swarms, n_part, seed)
            par_o = np.concatenate([po.to_params(x_o[s * n_part:(s + 1) * n_part], lo[s], hi[s]) for s in range(3)])
            F_o, _ = orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par_o)
            x, v, pb, pbf, fl = fs.fstat_pso_state(pso)
            np.testing.assert_array_equal(x, x_o)
            fin = np.isfinite(F_o)
            np.testing.assert_allclose(fl[fin], F_o[fin], rtol=1e-5)
            fs.fstat_pso_iterate(pso, n_iter)
            bp, bf = fs.fstat_pso_best(pso)
            x, v, pb, pbf, fl = fs.fstat_pso_state(pso)
            for s in range(3):
                assert np.all((bp[s] >= lo[s]) & (bp[s] <= hi[s]))
                sl = slice(s * n_part, (s + 1) * n_part)
                j = int(np.argmax(pbf[sl]))
                np.testing.assert_array_equal(bp[s], lo[s] + pb[sl][j] * (hi[s] - lo[s]))
                assert bf[s] == pbf[sl][j]
        with pytest.raises(fs.FstatError):
            fs.fstat_pso_create(plan, 3, 16, 4, hi, lo)


@pytest.mark.gpu
def test_many_iterations_without_host_sync_improve_every_swarm(gpu, orc):
    fs = gpu
    import torch
    year = 31557600.0
    cfg = syn.Config(16, "pso_slice2", 2.5 * year, 0.0200, 0.0202, (4,), (64,), 3.5 * year, "wide")
    ds = syn.make_dataset(cfg, orc.template, noise=False)
    inj = ds.inj_params
    lo = np.array([inj[0] - 2000.0, inj[1] * 0.999, 0.2, inj[3] - 0.05, inj[4] - 0.05, 0.0])
    hi = np.array([inj[0] + 2000.0, inj[1] * 1.001, 0.25, inj[3] + 0.05, inj[4] + 0.05, 0.1])
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(4)) as plan:
        F_inj, _ = fs.fstat_eval_batch_host(plan, inj[None, :])
        st = torch.cuda.Stream()
        with fs.fstat_pso_create(plan, 8, 128, 40, lo, hi, seed=7, stream=st) as pso:
            _, f0 = fs.fstat_pso_best(pso, stream=st)
            fs.fstat_pso_iterate(pso, 40, stream=st)            # 40 iterations enqueued back to back
            bp, bf = fs.fstat_pso_best(pso, stream=st)
            assert np.all(bf >= f0) and np.all(bf <= F_inj[0] * (1 + 1e-9))   # zero noise: F peaks at the injection
            assert np.all((bp >= lo) & (bp <= hi))
            assert (bf > f0).sum() >= 6
        with pytest.raises(fs.FstatError):
            fs.fstat_pso_create(plan, 0, 128, 40, lo, hi)
        with pytest.raises(fs.FstatError):
            fs.fstat_pso_create(plan, 1, 16, 10, hi, lo)


@pytest.mark.gpu
@pytest.mark.parametrize("lattice", [64, 1])
def test_device_swarms_with_the_papers_segment_limits_as_fitness(gpu, orc, lattice):
    """Rows f1 x f2: band_n_seg >= 1 makes the swarm's fitness fstat_eval_batch_bands (per-template bands,
    PAPER.md:122).  Same step-by-step bit-equality of the swarm state with the PSO oracle fed the device's F;
    the fitness itself against the oracle's fstat_bands at the first and last iteration."""
    fs = gpu
    ds = syn.make_dataset(syn.BANDS_SMALL, orc.template)
    inj = ds.inj_params
    lo = np.array([inj[0] - 3000.0, inj[1] * 0.998, 0.2, inj[3] - 0.1, inj[4] - 0.1, 0.0])
    hi = np.array([inj[0] + 3000.0, inj[1] * 1.002, 0.25, inj[3] + 0.1, inj[4] + 0.1, 0.1])
    n_swarms, n_part, n_iter, seed, n_seg = 2, 16, 6, 99, 4
    opts = fs.fstat_pso_default_options(band_n_seg=n_seg, band_lattice=lattice)
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(1)) as plan:
        with fs.fstat_pso_create(plan, n_swarms, n_part, n_iter, lo, hi, seed, opts) as pso:
            x_o, v_o = po.init(n_swarms, n_part, seed)
            x, v, pb, pf, fl = fs.fstat_pso_state(pso)
            np.testing.assert_array_equal(x, x_o)
            F_o, _, _ = orc.fstat_bands(ds.freq, ds.dw, ds.inv_sn, po.to_params(x_o, lo, hi), n_seg, lattice)
            assert np.max(np.abs(fl - F_o) / np.abs(F_o)) <= 1e-5
            pb_o, pf_o = x_o.copy(), fl.copy()
            for it in range(1, n_iter + 1):
                fs.fstat_pso_iterate(pso, 1)
                x, v, pb, pf, fl = fs.fstat_pso_state(pso)
                x_o, v_o = po.step(x_o, v_o, pb_o, pf_o, n_part, it, n_iter, seed)
                np.testing.assert_array_equal(x, x_o, err_msg="iteration %d" % it)
                np.testing.assert_array_equal(v, v_o)
                par_o = po.to_params(x_o, lo, hi)
                outside = np.isnan(par_o[:, 0])
                assert np.all(np.isneginf(fl[outside])) and np.all(np.isfinite(fl[~outside]))
                pb_o, pf_o = po.update_best(x_o, fl, pb_o, pf_o)
                np.testing.assert_array_equal(pf, pf_o)
            F_o, _, _ = orc.fstat_bands(ds.freq, ds.dw, ds.inv_sn, par_o[~outside], n_seg, lattice)
            assert np.max(np.abs(fl[~outside] - F_o) / np.abs(F_o)) <= 1e-5
