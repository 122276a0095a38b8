"""CPU oracle of the L1 + SSIM image loss -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it shares no code with
the CUDA path.  Plain numpy in float64, written as the definition.

The paper trains with the loss of its reference method [10] ("computes the loss"; refs [31] SSIM, [20]
fused SSIM): L = (1 - lambda) * mean|x - y| + lambda * (1 - mean SSIM(x, y)), lambda = 0.2, SSIM per channel with an
11 x 11 Gaussian window (sigma 1.5, normalised to sum 1), zero padding ("same" size), C1 = 0.01^2, C2 = 0.03^2,
means over all views, pixels and channels.  Readings (listed in DESIGN.md): biased (window-weighted) variances
s11 = E[x^2] - mu1^2; zero padding contributes zeros to every window sum (the window is NOT renormalised at the border).

Images are [C, H, W, 3] like the rasteriser's output.
"""
from __future__ import annotations

import numpy as np

WIN = 11
SIGMA = 1.5
C1 = 0.01 ** 2
C2 = 0.03 ** 2


def window_1d():
    """exp(-(k - 5)^2 / (2 sigma^2)), k = 0..10, normalised to sum 1; the 2-D window is its outer product."""
    k = np.arange(WIN, dtype=np.float64) - WIN // 2
    g = np.exp(-(k * k) / (2.0 * SIGMA * SIGMA))
    return g / g.sum()


def conv_same(img):
    """Direct 2-D correlation of every [H, W] slice of a [C, H, W, 3] array with the 11 x 11 window, zero padding."""
    g = window_1d()
    w2 = np.outer(g, g)
    C, H, W, ch = img.shape
    r = WIN // 2
    pad = np.zeros((C, H + 2 * r, W + 2 * r, ch), dtype=np.float64)
    pad[:, r:r + H, r:r + W, :] = img
    out = np.zeros((C, H, W, ch), dtype=np.float64)
    for dy in range(WIN):
        for dx in range(WIN):
            out += w2[dy, dx] * pad[:, dy:dy + H, dx:dx + W, :]
    return out


def ssim_map(x, y):
    """Per pixel and channel SSIM and the window statistics it is built from."""
    x = np.asarray(x, np.float64); y = np.asarray(y, np.float64)
    mu1, mu2 = conv_same(x), conv_same(y)
    s11 = conv_same(x * x) - mu1 * mu1
    s22 = conv_same(y * y) - mu2 * mu2
    s12 = conv_same(x * y) - mu1 * mu2
    A1 = 2.0 * mu1 * mu2 + C1
    A2 = 2.0 * s12 + C2
    B1 = mu1 * mu1 + mu2 * mu2 + C1
    B2 = s11 + s22 + C2
    S = (A1 * A2) / (B1 * B2)
    return S, dict(mu1=mu1, mu2=mu2, s11=s11, s22=s22, s12=s12, A1=A1, A2=A2, B1=B1, B2=B2)


def l1_ssim_loss(x, y, lam=0.2):
    """L = (1 - lam) mean|x - y| + lam (1 - mean SSIM)."""
    x = np.asarray(x, np.float64); y = np.asarray(y, np.float64)
    S, _ = ssim_map(x, y)
    return (1.0 - lam) * np.abs(x - y).mean() + lam * (1.0 - S.mean())


def l1_ssim_loss_grad(x, y, lam=0.2):
    """(L, dL/dx).  With e11 = E[x^2], e12 = E[xy] (linear in x^2, xy) and S = S(mu1, s11 = e11 - mu1^2, s12 = e12 - mu1 mu2):
    dS/ds11 = -S / B2, dS/ds12 = 2 A1 / (B1 B2), dS/dmu1|s = 2 mu2 A2 / (B1 B2) - 2 mu1 S / B1, and
    dL/dx = conv(w dS/dmu1_total) + 2 x conv(w dS/ds11) + y conv(w dS/ds12), w = -lam / n (the window is symmetric and the
    padding is zero, so the adjoint of the correlation is the same correlation), plus the L1 term (1 - lam) sign(x - y) / n."""
    x = np.asarray(x, np.float64); y = np.asarray(y, np.float64)
    n = x.size
    S, st = ssim_map(x, y)
    dS_ds11 = -S / st["B2"]
    dS_ds12 = 2.0 * st["A1"] / (st["B1"] * st["B2"])
    dS_dmu1 = 2.0 * st["mu2"] * st["A2"] / (st["B1"] * st["B2"]) - 2.0 * st["mu1"] * S / st["B1"]
    dS_dmu1_total = dS_dmu1 - 2.0 * st["mu1"] * dS_ds11 - st["mu2"] * dS_ds12
    w = -lam / n
    g = conv_same(w * dS_dmu1_total) + 2.0 * x * conv_same(w * dS_ds11) + y * conv_same(w * dS_ds12)
    g += (1.0 - lam) * np.sign(x - y) / n
    L = (1.0 - lam) * np.abs(x - y).mean() + lam * (1.0 - S.mean())
    return L, g
