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
