"""CPU oracle of the fused Adam step over the Gaussian parameter arrays -- TEST
INFRASTRUCTURE ONLY; plain numpy float64, shares no code with the CUDA path.

PAPER.md:82 / :309 mention the fused Adam of the reference implementation; no formula is printed.  Readings (DESIGN.md
A27-A28): A27 the update is Adam as published (Kingma & Ba) with bias correction and eps outside the square root,
no weight decay, no amsgrad:
    m <- b1 m + (1 - b1) g;  v <- b2 v + (1 - b2) g^2;  p <- p - lr * (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps);
A28 the "visible-only" variant updates exactly the rows of Gaussians with radius > 0 in at least one view of the batch and
leaves parameter and both moments of every other row untouched (no decay of the moments of invisible Gaussians).
"""
from __future__ import annotations

import numpy as np


def adam_step(p, g, m, v, lr, b1, b2, eps, t, visible=None):
    """Returns new (p, m, v); `visible` is an optional boolean [N] row mask (A28); t >= 1 is the step count."""
    p = np.asarray(p, np.float64); g = np.asarray(g, np.float64)
    m = np.asarray(m, np.float64); v = np.asarray(v, np.float64)
    m2 = b1 * m + (1.0 - b1) * g
    v2 = b2 * v + (1.0 - b2) * g * g
    mhat = m2 / (1.0 - b1 ** t)
    vhat = v2 / (1.0 - b2 ** t)
    p2 = p - lr * mhat / (np.sqrt(vhat) + eps)
    if visible is not None:
        mask = np.asarray(visible, bool).reshape((-1,) + (1,) * (p.ndim - 1))
        p2 = np.where(mask, p2, p); m2 = np.where(mask, m2, m); v2 = np.where(mask, v2, v)
    return p2, m2, v2
