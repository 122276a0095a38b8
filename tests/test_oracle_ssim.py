"""Pins of the L1 + SSIM oracle (oracle/ssim_oracle.py) against things other than itself: closed forms, invariants,
a brute-force per-pixel evaluation written with Python loops, a library correlation, and finite differences."""
import numpy as np
import pytest
from scipy import ndimage

from oracle import ssim_oracle as S


def rnd(shape, seed):
    return np.random.default_rng(seed).random(shape)


def test_window_is_the_normalised_gaussian():
    g = S.window_1d()
    assert g.shape == (11,) and abs(g.sum() - 1.0) < 1e-15
    assert np.allclose(g, g[::-1], rtol=0, atol=0)
    # ratio of neighbouring taps of exp(-k^2 / (2 * 1.5^2)): g[5] / g[4] = exp(1 / 4.5)
    assert abs(g[5] / g[4] - np.exp(1.0 / 4.5)) < 1e-14
    assert abs(g[5] / g[0] - np.exp(25.0 / 4.5)) < 1e-11


def test_conv_matches_library_correlation_with_zero_padding():
    x = rnd((2, 19, 23, 3), 1)
    got = S.conv_same(x)
    w2 = np.outer(S.window_1d(), S.window_1d())
    for c in range(2):
        for ch in range(3):
            ref = ndimage.correlate(x[c, :, :, ch], w2, mode="constant", cval=0.0)
            assert np.abs(got[c, :, :, ch] - ref).max() < 1e-14


def test_identical_images_have_ssim_one_and_loss_zero():
    x = rnd((1, 20, 17, 3), 2)
    m, _ = S.ssim_map(x, x)
    assert np.abs(m - 1.0).max() < 1e-12
    assert abs(S.l1_ssim_loss(x, x)) < 1e-12


def test_constant_images_closed_form_in_the_interior():
    a, b = 0.3, 0.7
    x = np.full((1, 30, 30, 3), a); y = np.full((1, 30, 30, 3), b)
    m, _ = S.ssim_map(x, y)
    want = (2 * a * b + S.C1) / (a * a + b * b + S.C1)        # variances and covariance vanish: the C2 factors cancel
    assert np.abs(m[:, 5:-5, 5:-5, :] - want).max() < 1e-12
    # at the corner the zero padding enters the window sums: mu = a * (partial window mass), not a
    g = S.window_1d()
    mass = g[5:].sum() ** 2
    mu1, mu2 = a * mass, b * mass
    s11, s22, s12 = a * a * mass - mu1 ** 2, b * b * mass - mu2 ** 2, a * b * mass - mu1 * mu2
    corner = ((2 * mu1 * mu2 + S.C1) * (2 * s12 + S.C2)) / ((mu1 ** 2 + mu2 ** 2 + S.C1) * (s11 + s22 + S.C2))
    assert abs(m[0, 0, 0, 0] - corner) < 1e-12


def test_symmetry_and_flip_invariance():
    x, y = rnd((1, 16, 21, 3), 3), rnd((1, 16, 21, 3), 4)
    mxy, _ = S.ssim_map(x, y)
    myx, _ = S.ssim_map(y, x)
    assert np.abs(mxy - myx).max() < 1e-13
    mf, _ = S.ssim_map(x[:, ::-1, ::-1], y[:, ::-1, ::-1])
    assert np.abs(mf[:, ::-1, ::-1] - mxy).max() < 1e-13
    assert abs(S.l1_ssim_loss(x, y) - S.l1_ssim_loss(np.swapaxes(x, 1, 2), np.swapaxes(y, 1, 2))) < 1e-13


def test_brute_force_per_pixel_loops():
    """Every pixel's SSIM from explicit loops over its 11 x 11 neighbourhood (independent of conv_same)."""
    x, y = rnd((1, 9, 8, 3), 5), rnd((1, 9, 8, 3), 6)
    g = S.window_1d()
    H, W = 9, 8
    m, _ = S.ssim_map(x, y)
    for i in range(H):
        for j in range(W):
            for ch in range(3):
                mu1 = mu2 = e11 = e22 = e12 = 0.0
                for dy in range(-5, 6):
                    for dx in range(-5, 6):
                        ii, jj = i + dy, j + dx
                        if 0 <= ii < H and 0 <= jj < W:
                            w = g[dy + 5] * g[dx + 5]
                            a, b = x[0, ii, jj, ch], y[0, ii, jj, ch]
                            mu1 += w * a; mu2 += w * b; e11 += w * a * a; e22 += w * b * b; e12 += w * a * b
                s11, s22, s12 = e11 - mu1 * mu1, e22 - mu2 * mu2, e12 - mu1 * mu2
                want = ((2 * mu1 * mu2 + S.C1) * (2 * s12 + S.C2)) / ((mu1 * mu1 + mu2 * mu2 + S.C1) * (s11 + s22 + S.C2))
                assert abs(m[0, i, j, ch] - want) < 1e-12
    L = 0.8 * np.abs(x - y).mean() + 0.2 * (1.0 - m.mean())
    assert abs(S.l1_ssim_loss(x, y) - L) < 1e-15


@pytest.mark.parametrize("lam", [0.2, 1.0, 0.0])
def test_gradient_against_central_differences(lam):
    x, y = rnd((2, 13, 12, 3), 7), rnd((2, 13, 12, 3), 8)
    L, g = S.l1_ssim_loss_grad(x, y, lam)
    assert abs(L - S.l1_ssim_loss(x, y, lam)) < 1e-15
    rng = np.random.default_rng(9)
    h = 1e-6
    for _ in range(40):
        idx = tuple(rng.integers(0, s) for s in x.shape)
        if abs(x[idx] - y[idx]) < 10 * h:
            continue                                        # the L1 term is not differentiable at x = y
        xp, xm = x.copy(), x.copy()
        xp[idx] += h; xm[idx] -= h
        fd = (S.l1_ssim_loss(xp, y, lam) - S.l1_ssim_loss(xm, y, lam)) / (2 * h)
        assert abs(fd - g[idx]) <= 1e-7 * max(1.0, abs(fd) * 1e3), (idx, fd, g[idx])


def test_gradient_directional_derivative_whole_image():
    x, y = rnd((1, 24, 20, 3), 10), rnd((1, 24, 20, 3), 11)
    _, g = S.l1_ssim_loss_grad(x, y, 1.0)                   # SSIM term only (smooth everywhere)
    d = np.random.default_rng(12).standard_normal(x.shape)
    h = 1e-6
    fd = (S.l1_ssim_loss(x + h * d, y, 1.0) - S.l1_ssim_loss(x - h * d, y, 1.0)) / (2 * h)
    assert abs(fd - (g * d).sum()) <= 1e-8 * max(1.0, abs(fd))
