"""CPU oracle of the 3-D Morton ordering of the Gaussian arrays -- TEST INFRASTRUCTURE ONLY.

PAPER.md:217: the Gaussians are "sorted along a Morton curve" so that Gaussians that are close in space are close in
memory.  The paper gives no bit layout; readings (A24-A26):
  A24  every coordinate is quantised to 21 bits over the bounding box [lo, hi] of the means:
       q = clamp(floor((p - lo) * scale), 0, 2^21 - 1),  scale = 2^21 / (hi - lo)   (1 when hi == lo),
       evaluated in fp32 with one rounding per operation (the quantisation decides integers, so both sides use the
       kernel's precision);
  A25  code = interleave(qx, qy, qz): bit k of qx -> bit 3k+2, of qy -> bit 3k+1, of qz -> bit 3k  (63 bits, x most significant);
  A26  the order is the stable ascending order of the codes (ties keep ascending index).
Plain numpy; shares no code with the CUDA path.
"""
from __future__ import annotations

import numpy as np

BITS = 21


def bounds(means):
    means = np.asarray(means, np.float32)
    return means.min(axis=0).astype(np.float32), means.max(axis=0).astype(np.float32)


def scales(lo, hi):
    """fp32: 2^21 / (hi - lo) per axis, 1 for a degenerate axis."""
    lo = np.asarray(lo, np.float32); hi = np.asarray(hi, np.float32)
    ext = (hi - lo).astype(np.float32)
    out = np.ones(3, np.float32)
    nz = ext > 0
    out[nz] = (np.float32(2 ** BITS) / ext[nz]).astype(np.float32)
    return out


def quantise(means, lo, hi):
    means = np.asarray(means, np.float32)
    lo = np.asarray(lo, np.float32)
    sc = scales(lo, hi)
    t = ((means - lo).astype(np.float32) * sc).astype(np.float32)       # one rounding per operation
    q = np.floor(t)
    q = np.where(np.isfinite(q), q, 0.0)
    return np.clip(q, 0, 2 ** BITS - 1).astype(np.uint64)


def interleave(q):
    """[N, 3] 21-bit integers -> [N] 63-bit codes, bit by bit."""
    q = np.asarray(q, np.uint64)
    code = np.zeros(q.shape[0], np.uint64)
    for k in range(BITS):
        for axis, off in ((0, 2), (1, 1), (2, 0)):
            bit = (q[:, axis] >> np.uint64(k)) & np.uint64(1)
            code |= bit << np.uint64(3 * k + off)
    return code


def morton_codes(means, lo=None, hi=None):
    if lo is None or hi is None:
        lo, hi = bounds(means)
    return interleave(quantise(means, lo, hi))


def morton_order(means, lo=None, hi=None):
    """Permutation perm with codes[perm] ascending, ties in ascending index."""
    return np.argsort(morton_codes(means, lo, hi), kind="stable").astype(np.int32)
