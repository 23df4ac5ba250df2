"""CPU oracle of the PSO update (Sec. III.A; Eq. 13-14 :146-150).  TEST INFRASTRUCTURE ONLY:
nothing of the product path may import this module, and it imports nothing of the product.

Plain numpy, one statement per step of the paper's description:
  * x ~ U[a, b], v ~ U[a - x, b - x] at the start (:158), in the unit box;
  * lbest ring topology: the best personal best among the neighbours i-1, i, i+1 (:152);
  * v <- w v + c1 r1 (pbest - x) + c2 r2 (lbest - x), |v| <= v_max; x <- x + v (Eq. 13-14; reading A20);
  * inertia w falling linearly from w_start to w_end over the run; c1 = c2 = 2, v_max = 0.5 (:162);
  * "let them fly": a particle outside the box is not evaluated and has fitness -inf (:158);
  * a personal best is replaced only by a strictly larger fitness.
The paper names no random-number generator.  Both sides draw from Philox4x32-10 (Salmon et al., SC'11) with
counter (particle, iteration, draw, 0) and key = seed; uniform = (uint32 + 0.5) / 2^32; draws 0..5 are r1 (or the
initial x), 6..11 r2 (or the initial v draw).  The generator is pinned by the Random123 known-answer vectors in
tests/golden/philox4x32_10_kat.json.  The floating-point order of Eq. 14 is ((w v) + ((c1 r1)(pbest - x))) +
((c2 r2)(lbest - x)), every product and sum rounded to nearest separately.
"""
from __future__ import annotations

import numpy as np

_M0, _M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_W0, _W1 = 0x9E3779B9, 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Ten rounds of Philox-4x32 on arrays of uint32 counters / keys; returns four uint32 arrays."""
    c = [np.asarray(x, dtype=np.uint64) & _MASK for x in np.broadcast_arrays(c0, c1, c2, c3)]
    k0 = int(k0) & 0xFFFFFFFF
    k1 = int(k1) & 0xFFFFFFFF
    for _ in range(10):
        p0, p1 = _M0 * c[0], _M1 * c[2]
        c = [((p1 >> np.uint64(32)) ^ c[1] ^ np.uint64(k0)) & _MASK, p1 & _MASK,
             ((p0 >> np.uint64(32)) ^ c[3] ^ np.uint64(k1)) & _MASK, p0 & _MASK]
        k0 = (k0 + _W0) & 0xFFFFFFFF
        k1 = (k1 + _W1) & 0xFFFFFFFF
    return [x.astype(np.uint32) for x in c]


def uniforms12(n: int, iteration: int, seed: int) -> np.ndarray:
    """[n][12] uniforms in (0, 1) of the particles 0..n-1 at one iteration."""
    gid = np.arange(n, dtype=np.uint64)
    out = np.empty((n, 12))
    for j in range(3):
        words = philox4x32_10(gid, np.uint64(iteration), np.uint64(j), np.uint64(0), seed & 0xFFFFFFFF, seed >> 32)
        for q in range(4):
            out[:, 4 * j + q] = (words[q].astype(np.float64) + 0.5) * 2.3283064365386963e-10
    return out


def init(n_swarms: int, n_particles: int, seed: int, v_max: float = 0.5):
    """(x, v) [N][6] of the initial swarms, N = n_swarms * n_particles."""
    u = uniforms12(n_swarms * n_particles, 0, seed)
    x = u[:, :6].copy()
    v = np.clip(u[:, 6:] - x, -v_max, v_max)
    return x, v


def to_params(x: np.ndarray, lo, hi) -> np.ndarray:
    """Physical parameters lo + x (hi - lo); NaN rows for particles outside the unit box (not evaluated)."""
    lo, hi = np.asarray(lo, dtype=np.float64), np.asarray(hi, dtype=np.float64)
    par = lo + x * (hi - lo)
    par[~np.all((x >= 0.0) & (x <= 1.0), axis=1)] = np.nan
    return par


def inertia(iteration: int, n_iter_total: int, w_start: float = 0.9, w_end: float = 0.4) -> float:
    frac = (iteration - 1) / float(max(n_iter_total - 1, 1))
    return w_start + (w_end - w_start) * min(frac, 1.0)


def step(x, v, pbest, pbest_f, n_particles: int, iteration: int, n_iter_total: int, seed: int, c1: float = 2.0,
         c2: float = 2.0, v_max: float = 0.5, w_start: float = 0.9, w_end: float = 0.4):
    """One iteration (1-based) of Eq. 13-14 for all swarms; returns the new (x, v)."""
    n = x.shape[0]
    n_swarms = n // n_particles
    f = pbest_f.reshape(n_swarms, n_particles)
    stack = np.stack([np.roll(f, 1, axis=1), f, np.roll(f, -1, axis=1)])      # left, self, right
    who = np.argmax(stack, axis=0) - 1                                        # first maximum in that order
    idx = (np.arange(n_particles)[None, :] + who) % n_particles
    lbest = np.take_along_axis(pbest.reshape(n_swarms, n_particles, 6), idx[:, :, None], axis=1).reshape(n, 6)
    u = uniforms12(n, iteration, seed)
    w = inertia(iteration, n_iter_total, w_start, w_end)
    vn = ((w * v) + ((c1 * u[:, :6]) * (pbest - x))) + ((c2 * u[:, 6:]) * (lbest - x))
    vn = np.clip(vn, -v_max, v_max)
    return x + vn, vn


def update_best(x, f, pbest, pbest_f):
    better = f > pbest_f
    pbest = pbest.copy()
    pbest_f = pbest_f.copy()
    pbest[better] = x[better]
    pbest_f[better] = f[better]
    return pbest, pbest_f
