"""The thin host PSO loop (Eq. 13-14): CPU tests of the update rule with analytic fitness
functions, and one GPU test that drives fstat_eval_batch with several batched swarms."""
import numpy as np
import pytest

import synthetic as syn
from paper_2407_10797_b200.pso import pso_maximise


def _sphere(centre):
    def f(par):
        out = -np.sum((par - centre) ** 2, axis=1)
        out[np.isnan(out)] = -np.inf                      # what the library does for NaN rows
        return out
    return f


def test_pso_finds_the_maximum_of_a_smooth_function_and_is_reproducible():
    lo, hi = np.zeros(6), np.array([1.0, 2.0, 3.0, 4.0, 5.0, 6.0])
    centre = lo + 0.37 * (hi - lo)
    best, fbest, hist = pso_maximise(_sphere(centre), lo, hi, n_swarms=3, n_particles=32, n_iter=200, seed=5)
    assert best.shape == (3, 6) and fbest.shape == (3,) and hist.shape == (201, 3)
    assert np.all(np.diff(hist, axis=0) >= 0.0)           # swarm-best fitness never decreases
    assert np.all(fbest > -1e-3) and np.allclose(best, centre, atol=0.05)
    best2, fbest2, _ = pso_maximise(_sphere(centre), lo, hi, n_swarms=3, n_particles=32, n_iter=200, seed=5)
    np.testing.assert_array_equal(best, best2)
    np.testing.assert_array_equal(fbest, fbest2)


def test_particles_outside_the_box_are_not_evaluated():
    """Let them fly: rows outside the box reach the fitness function as NaN."""
    seen = {"nan_rows": 0, "calls": 0}

    def f(par):
        bad = np.isnan(par).any(axis=1)
        seen["nan_rows"] += int(bad.sum())
        seen["calls"] += 1
        good = par[~bad]
        assert np.all(good >= 0.0) and np.all(good <= 1.0)
        out = -np.sum((par - 0.95) ** 2, axis=1)          # maximum near a corner: particles overshoot the box
        out[bad] = -np.inf
        return out
    best, fbest, hist = pso_maximise(f, np.zeros(6), np.ones(6), n_swarms=1, n_particles=16, n_iter=60, seed=1)
    assert seen["calls"] == 61 and seen["nan_rows"] > 0
    assert np.all((best >= 0.0) & (best <= 1.0)) and np.isfinite(fbest).all()


@pytest.mark.gpu
def test_batched_swarms_drive_the_library(orc):
    """8 independent swarms of 32 particles in ONE fstat_eval_batch call per iteration, on a zero-noise
    fine-grid slice with an injection: every swarm's best F grows and ends above the typical noise-free
    off-signal value; out-of-box particles (NaN rows) come back as -inf from the library."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2407_10797_b200 as fs
    from paper_2407_10797_b200.pso import fstat_fitness
    year = 31557600.0
    cfg = syn.Config(12, "pso_slice", 2.5 * year, 0.0200, 0.0202, (4,), (256,), 3.5 * year, "wide")
    ds = syn.make_dataset(cfg, orc.template, noise=False)
    inj = ds.inj_params
    lo = np.array([inj[0] - 2000.0, inj[1] * 0.999, 0.2, inj[3] - 0.05, inj[4] - 0.05, 0.0])
    hi = np.array([inj[0] + 2000.0, inj[1] * 1.001, 0.25, inj[3] + 0.05, inj[4] + 0.05, 0.1])
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, ds.edges(4)) as plan:
        fit = fstat_fitness(plan)
        probe = np.vstack([inj, np.full(6, np.nan)])
        f_probe = fit(probe)
        assert np.isneginf(f_probe[1]) and f_probe[0] > 0.0
        best, fbest, hist = pso_maximise(fit, lo, hi, n_swarms=8, n_particles=32, n_iter=25, seed=2)
        assert np.all(np.diff(hist, axis=0) >= 0.0)
        assert np.all(fbest >= hist[0])
        assert np.all(fbest <= f_probe[0] * (1.0 + 1e-9))  # zero noise: F peaks at the injected parameters
        assert (fbest > hist[0]).any()                     # the swarms do climb
        assert fs.fstat_plan_launch_count(plan) > 0
