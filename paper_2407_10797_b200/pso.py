"""Thin host PSO loop driving the batched F-statistic (§III.A; Eq. 13-14 :146-150).

Not on the hot path and not a search pipeline: it is the example driver north_star names, used to show how a
swarm (or several independent swarms batched in ONE call) talks to ``fstat_eval_batch``.
Settings follow the paper: lbest ring topology, c1 = c2 = 2, |v| <= v_max = 0.5 in box units, linearly decaying
inertia, "let them fly" (particles outside the box keep moving and get fitness -inf without being evaluated:
here their parameters are sent as NaN, which the library maps to F = -inf), a fixed number of
iterations.  Positions live in the unit box [0, 1]^6 and are mapped to (t_c, M_c, eta, theta, phi, e0).
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple

import numpy as np


def pso_maximise(fitness: Callable[[np.ndarray], np.ndarray], lo, hi, n_swarms: int = 1, n_particles: int = 128,
                 n_iter: int = 100, seed: int = 0, c1: float = 2.0, c2: float = 2.0, v_max: float = 0.5,
                 w_start: float = 0.9, w_end: float = 0.4) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Maximise ``fitness`` over the box [lo, hi] with ``n_swarms`` independent lbest swarms.

    ``fitness(params[n, d]) -> F[n]`` is called once per iteration with the particles of ALL swarms
    (rows outside the box are NaN and must come back as -inf).  Returns (best_params[n_swarms, d],
    best_fitness[n_swarms], history[n_iter + 1, n_swarms] of the swarm-best fitness)."""
    lo = np.asarray(lo, dtype=np.float64)
    hi = np.asarray(hi, dtype=np.float64)
    d = lo.shape[0]
    rng = np.random.default_rng(seed)
    x = rng.uniform(0.0, 1.0, (n_swarms, n_particles, d))                 # x ~ U[a, b]           (:158)
    v = rng.uniform(0.0, 1.0, (n_swarms, n_particles, d)) - x             # v ~ U[a - x, b - x]   (:158)
    v = np.clip(v, -v_max, v_max)

    def evaluate(pos):
        inside = np.all((pos >= 0.0) & (pos <= 1.0), axis=2)
        par = lo + pos * (hi - lo)
        par[~inside] = np.nan                                              # let them fly: not evaluated
        f = np.asarray(fitness(par.reshape(-1, d)), dtype=np.float64).reshape(n_swarms, n_particles)
        f[~inside] = -np.inf
        return f

    f = evaluate(x)
    pbest, pbest_f = x.copy(), f.copy()
    history = np.empty((n_iter + 1, n_swarms))
    history[0] = pbest_f.max(axis=1)
    for it in range(n_iter):
        # lbest: best personal best among the ring neighbours i-1, i, i+1
        stack = np.stack([np.roll(pbest_f, 1, axis=1), pbest_f, np.roll(pbest_f, -1, axis=1)])
        who = np.argmax(stack, axis=0) - 1                                 # -1, 0, +1
        idx = (np.arange(n_particles)[None, :] + who) % n_particles
        lbest = np.take_along_axis(pbest, idx[:, :, None], axis=1)
        w = w_start + (w_end - w_start) * it / max(n_iter - 1, 1)
        r1 = rng.uniform(0.0, 1.0, x.shape)
        r2 = rng.uniform(0.0, 1.0, x.shape)
        v = w * v + c1 * r1 * (pbest - x) + c2 * r2 * (lbest - x)          # Eq. 14 :150
        v = np.clip(v, -v_max, v_max)                                      # reading A20: clamp |v|
        x = x + v                                                          # Eq. 13 :146
        f = evaluate(x)
        better = f > pbest_f
        pbest[better] = x[better]
        pbest_f[better] = f[better]
        history[it + 1] = pbest_f.max(axis=1)
    best = np.argmax(pbest_f, axis=1)
    best_pos = pbest[np.arange(n_swarms), best]
    return lo + best_pos * (hi - lo), pbest_f[np.arange(n_swarms), best], history


def fstat_fitness(plan, stream=None) -> Callable[[np.ndarray], np.ndarray]:
    """Fitness callback that evaluates F for a batch of parameter rows through ``fstat_eval_batch_host``."""
    from . import binding

    def fn(par: np.ndarray) -> np.ndarray:
        F, _ = binding.fstat_eval_batch_host(plan, np.ascontiguousarray(par, dtype=np.float64), want_Fk=False,
                                             stream=stream)
        return F
    return fn
