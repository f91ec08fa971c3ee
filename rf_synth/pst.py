"""Pre-sampled Particle Swarm Template (PST): N i.i.d. points uniform in the unit 6-D ball.

PAPER.md L190 ("pre-sample a fixed number of particles uniformly within the unit sphere in the 6D
state space"); BASELINE.json configs ("uniform in the unit 6D ball").  The PST is an *input* of the
method (Algorithm 1, "Input: ... Pre-sampled PST"), handed unchanged to the oracle and the CUDA
path.  Direction = normalised 6-D Gaussian, radius = U^(1/6)  (radial CDF r^6).
"""
from __future__ import annotations

import numpy as np


def sample_pst(n: int, seed: int) -> np.ndarray:
    """(n, 6) float32, every row with Euclidean norm <= 1 (also after rounding to float32)."""
    rng = np.random.Generator(np.random.Philox(int(seed)))
    g = rng.standard_normal((n, 6))
    u = rng.random(n)
    p = g / np.linalg.norm(g, axis=1, keepdims=True) * (u ** (1.0 / 6.0))[:, None]
    p32 = p.astype(np.float32)
    # float32 rounding can push a norm a hair above 1; pull such rows back inside the ball.
    nrm = np.linalg.norm(p32.astype(np.float64), axis=1)
    over = nrm > 1.0
    if np.any(over):
        p32[over] = (p32[over].astype(np.float64) * (1.0 - 1e-6) / nrm[over, None]).astype(np.float32)
    return np.ascontiguousarray(p32)


def sample_pst_poisson(n: int, seed: int, return_radius: bool = False):
    """(n, 6) float32 Poisson-disk ("blue noise") PST in the unit 6-D ball: no two particles closer than a radius r.

    PAPER.md L284: "To realize an unbiased particle sampling, we adopt the 6D Poisson disk sampling proposed in
    [Bridson 2007]."  The paper gives no radius; here r starts at the value at which random sequential addition
    still finds room for n points (2 (eta / n)^(1/6), eta = 0.06 of the ball's volume covered by the r/2-balls) and is
    relaxed by 3 % whenever 4000 consecutive darts are rejected, so the generator always terminates with exactly n
    points.  Dart throwing against all accepted points (O(n^2), a few seconds at n = 10240); like every generator in
    this package it is an INPUT recipe shared by the oracle and the CUDA path and holds none of the method's arithmetic.
    The guaranteed minimum distance (the smallest r used) is returned with return_radius=True."""
    rng = np.random.Generator(np.random.Philox(int(seed)))
    r = 2.0 * (0.06 / max(n, 1)) ** (1.0 / 6.0)
    pts = np.empty((n, 6), dtype=np.float64)
    count, rejected, r_min = 0, 0, r
    while count < n:
        g = rng.standard_normal((256, 6))
        cand = g / np.linalg.norm(g, axis=1, keepdims=True) * (rng.random(256) ** (1.0 / 6.0))[:, None] * (1.0 - 1e-6)
        for c in cand:
            if count == 0 or np.min(np.sum((pts[:count] - c) ** 2, axis=1)) >= r * r:
                pts[count] = c
                count += 1
                rejected = 0
                if count == n:
                    break
            else:
                rejected += 1
                if rejected >= 4000:
                    r *= 0.97
                    r_min = r
                    rejected = 0
    p32 = np.ascontiguousarray(pts.astype(np.float32))
    return (p32, float(r_min) * (1.0 - 1e-6)) if return_radius else p32
