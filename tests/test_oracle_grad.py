"""Pins for the oracle's backward stages O-R2 and O-P5:
central finite differences in double precision on tiny scenes (north_star), in "smooth mode"
(thresholds off) and in default mode guarded by an unchanged decision trace; linearity in
dL/dimage; exact zero gradient for culled Gaussians.
"""
import numpy as np
import pytest

from paper_2606_11390_b200 import scenes


def _small_scene(n=14, seed=11, deg=3):
    rng = np.random.default_rng(seed)
    K = (deg + 1) ** 2
    sc = {
        "means": rng.uniform(-0.8, 0.8, (n, 3)),
        "log_scales": rng.normal(-1.6, 0.4, (n, 3)),
        "quats": rng.standard_normal((n, 4)) * rng.uniform(0.5, 2.0, (n, 1)),      # unnormalised (reading A1)
        "opacity_logits": rng.normal(0.0, 1.0, n),
        "sh": np.concatenate([rng.normal(0, 0.5, (n, 1, 3)), rng.normal(0, 0.3, (n, K - 1, 3))], axis=1),
        "sh_degree": deg,
        "bg": np.array([0.3, 0.1, 0.2]),
    }
    sc["cameras"] = [
        scenes.make_camera(32, 24, 30.0, 28.0, (0.4, -0.3, -3.0), (0.1, 0.0, 0.0), (0.05, -1, 0.1), cx=15.0, cy=12.5),
        scenes.make_camera(32, 24, 30.0, 28.0, (2.5, 0.6, -1.5), (0.0, 0.1, 0.0), (0, -1, 0)),
    ]
    # one Gaussian far off-axis so that the Jacobian clamp of O-P1 step 3 is active in camera 0
    sc["means"][0] = [2.6, 0.2, 0.3]
    sc["log_scales"][0] = [-0.3, -0.5, -0.4]
    # one Gaussian with a negative (clamped) colour channel
    sc["sh"][1, 0, 0] = -4.0
    return sc


def _forward_f64(oracle, cfg, sc):
    """Whole forward in double with NO fp32 rounding of the stage hand-off (for finite differences)."""
    cams = sc["cameras"]
    pf = oracle.project_fwd(cfg, sc["means"], sc["log_scales"], sc["quats"], sc["opacity_logits"], sc["sh"], cams)
    keys, vals, ranges = oracle.bin_tiles(cfg, cams, pf["means2d"], pf["depths"], pf["radii"])
    img, T, nc = oracle.raster_fwd(cfg, cams, vals, ranges, pf["means2d"], pf["conics"], pf["opacities"], pf["rgbs"], sc["bg"])
    return pf, vals, ranges, img, T, nc


def _backward_f64(oracle, cfg, sc, wimg):
    pf, vals, ranges, img, T, nc = _forward_f64(oracle, cfg, sc)
    g2 = oracle.raster_bwd(cfg, sc["cameras"], vals, ranges, pf["means2d"], pf["conics"], pf["opacities"], pf["rgbs"],
                           sc["bg"], T, nc, wimg)
    gp = oracle.project_bwd(cfg, sc["means"], sc["log_scales"], sc["quats"], sc["opacity_logits"], sc["sh"],
                            sc["cameras"], pf["radii"], g2["means2d"], g2["conics"], g2["opacities"], g2["rgbs"])
    return pf, g2, gp, (vals, ranges, nc)


def _loss(oracle, cfg, sc, wimg):
    return float((_forward_f64(oracle, cfg, sc)[3] * wimg).sum())


def _fd_check(oracle, cfg, sc, wimg, gp, names, per_tensor=40, h=1e-6, rtol=2e-6, trace=None):
    rng = np.random.default_rng(5)
    worst = 0.0
    for name in names:
        arr = sc[name]
        flat_idx = rng.choice(arr.size, size=min(per_tensor, arr.size), replace=False)
        num = np.zeros(len(flat_idx)); ana = np.zeros(len(flat_idx))
        for k, fi in enumerate(flat_idx):
            idx = np.unravel_index(fi, arr.shape)
            old = arr[idx]
            arr[idx] = old + h
            if trace is not None:
                assert trace(sc), f"decision trace changed at {name}{idx} (+h)"
            lp = _loss(oracle, cfg, sc, wimg)
            arr[idx] = old - h
            if trace is not None:
                assert trace(sc), f"decision trace changed at {name}{idx} (-h)"
            lm = _loss(oracle, cfg, sc, wimg)
            arr[idx] = old
            num[k] = (lp - lm) / (2 * h)
            ana[k] = gp[name][idx]
        scale = max(np.abs(num).max(), 1e-12)
        err = np.abs(num - ana).max() / scale
        worst = max(worst, err)
        assert err < rtol, f"{name}: FD mismatch {err:.3e}\nnum={num}\nana={ana}"
        assert np.abs(ana).max() > 0, f"{name}: gradient identically zero on the sampled entries"
    return worst


def test_smooth_mode_parameter_gradients_match_finite_differences(oracle):
    sc = _small_scene()
    cfg = oracle.smooth_cfg(sh_degree=3)
    wimg = np.random.default_rng(3).standard_normal((2, 24, 32, 3))
    pf, g2, gp, _ = _backward_f64(oracle, cfg, sc, wimg)
    assert np.all(pf["radii"] > 0)
    _fd_check(oracle, cfg, sc, wimg, gp, ["means", "log_scales", "quats", "opacity_logits", "sh"])


def test_smooth_mode_jacobian_clamp_branch_is_exercised(oracle):
    sc = _small_scene()
    cfg = oracle.smooth_cfg(sh_degree=3)
    cam = sc["cameras"][0]
    vm = cam["viewmat"]
    t = vm[:, :3] @ sc["means"][0] + vm[:, 3]
    assert abs(t[0] / t[2]) > 1.3 * cam["width"] / (2 * cam["fx"])      # clamp active for Gaussian 0 in camera 0
    wimg = np.random.default_rng(4).standard_normal((2, 24, 32, 3))
    _, _, gp, _ = _backward_f64(oracle, cfg, sc, wimg)
    rng = np.random.default_rng(0)
    # finite differences on exactly that Gaussian's parameters
    for name in ("means", "log_scales", "quats"):
        for j in range(sc[name].shape[1]):
            h = 1e-6
            old = sc[name][0, j]
            sc[name][0, j] = old + h; lp = _loss(oracle, cfg, sc, wimg)
            sc[name][0, j] = old - h; lm = _loss(oracle, cfg, sc, wimg)
            sc[name][0, j] = old
            num = (lp - lm) / (2 * h)
            assert abs(num - gp[name][0, j]) <= 2e-6 * max(1.0, abs(num)), (name, j, num, gp[name][0, j])


def test_smooth_mode_raster_gradients_match_finite_differences(oracle):
    """O-R2 alone: differentiate the image with respect to the projected 2-D records."""
    sc = _small_scene()
    cfg = oracle.smooth_cfg(sh_degree=3)
    cams = sc["cameras"]
    pf, vals, ranges, img, T, nc = _forward_f64(oracle, cfg, sc)
    wimg = np.random.default_rng(8).standard_normal(img.shape)
    g2 = oracle.raster_bwd(cfg, cams, vals, ranges, pf["means2d"], pf["conics"], pf["opacities"], pf["rgbs"], sc["bg"], T, nc, wimg)
    rec = {k: pf[k].copy() for k in ("means2d", "conics", "opacities", "rgbs")}

    def loss():
        im = oracle.raster_fwd(cfg, cams, vals, ranges, rec["means2d"], rec["conics"], rec["opacities"], rec["rgbs"], sc["bg"])[0]
        return float((im * wimg).sum())

    rng = np.random.default_rng(9)
    for name in rec:
        arr = rec[name]
        for fi in rng.choice(arr.size, size=min(30, arr.size), replace=False):
            idx = np.unravel_index(fi, arr.shape)
            h = 1e-6 * max(1.0, abs(arr[idx]))
            old = arr[idx]
            arr[idx] = old + h; lp = loss()
            arr[idx] = old - h; lm = loss()
            arr[idx] = old
            num = (lp - lm) / (2 * h)
            assert abs(num - g2[name][idx]) <= 5e-7 * max(1.0, abs(num)), (name, idx, num, g2[name][idx])


def test_default_mode_gradients_match_finite_differences_with_unchanged_decisions(oracle):
    """Default thresholds (alpha_min, alpha_max, t_min, 3-sigma extent): finite differences are
    valid wherever the piecewise-constant decisions (radii, tile lists, n_contrib) do not move."""
    sc = _small_scene(n=40, seed=21)
    sc["log_scales"] -= 1.0
    sc["opacity_logits"] += 2.5                      # several alphas hit the 0.99 clamp and pixels saturate
    cfg = oracle.make_cfg(sh_degree=3)
    wimg = np.random.default_rng(6).standard_normal((2, 24, 32, 3))
    pf, g2, gp, (vals0, ranges0, nc0) = _backward_f64(oracle, cfg, sc, wimg)
    assert (pf["radii"] == 0).any() and (pf["radii"] > 0).sum() > 20
    assert (nc0 < (ranges0[:, 1] - ranges0[:, 0]).max()).any()

    def trace(s):
        pf1, vals1, ranges1, _, _, nc1 = _forward_f64(oracle, cfg, s)
        return (np.array_equal(pf1["radii"], pf["radii"]) and np.array_equal(vals1, vals0)
                and np.array_equal(ranges1, ranges0) and np.array_equal(nc1, nc0))

    # per-entry skip decisions (alpha < 1/255, clamp) can still flip inside a pixel; h is small enough that
    # this did not happen for the sampled entries (a flip would show up as an O(1) mismatch)
    _fd_check(oracle, cfg, sc, wimg, gp, ["means", "log_scales", "quats", "opacity_logits", "sh"],
              per_tensor=25, h=1e-7, rtol=2e-5, trace=trace)


def test_gradients_are_linear_in_dL_dimage_and_zero_for_culled(oracle):
    sc = _small_scene(n=30, seed=5)
    sc["means"][3] = [0.0, 0.0, -10.0]               # behind the cameras -> culled everywhere
    sc["means"][4] = [50.0, 0.0, 0.0]                # far off-screen -> no tiles
    cfg = oracle.make_cfg(sh_degree=3)
    rng = np.random.default_rng(2)
    w1 = rng.standard_normal((2, 24, 32, 3)); w2 = rng.standard_normal((2, 24, 32, 3))
    pf, _, g1, _ = _backward_f64(oracle, cfg, sc, w1)
    _, _, g2, _ = _backward_f64(oracle, cfg, sc, w2)
    _, _, g12, _ = _backward_f64(oracle, cfg, sc, 2.0 * w1 - 0.5 * w2)
    assert pf["radii"][0, 3] == 0 and pf["radii"][1, 3] == 0
    for name in g1:
        np.testing.assert_allclose(g12[name], 2.0 * g1[name] - 0.5 * g2[name], rtol=1e-9, atol=1e-12)
        for i in (3, 4):
            if np.all(pf["radii"][:, i] == 0):
                assert np.all(g1[name][i] == 0)
    assert np.all(pf["radii"][:, 3] == 0)


def test_project_bwd_accumulate_flag(oracle):
    sc = _small_scene(n=10, seed=1)
    cfg = oracle.make_cfg(sh_degree=3)
    w = np.random.default_rng(1).standard_normal((2, 24, 32, 3))
    pf, g2, gp, _ = _backward_f64(oracle, cfg, sc, w)
    acc = {k: np.ones_like(v) for k, v in gp.items()}
    oracle.project_bwd(cfg, sc["means"], sc["log_scales"], sc["quats"], sc["opacity_logits"], sc["sh"], sc["cameras"],
                       pf["radii"], g2["means2d"], g2["conics"], g2["opacities"], g2["rgbs"], accumulate_into=acc)
    for k in gp:
        np.testing.assert_allclose(acc[k], gp[k] + 1.0, rtol=1e-13)


def test_views_sum_in_project_bwd(oracle):
    """a Gaussian visible in several cameras receives the sum of their contributions."""
    sc = _small_scene(n=12, seed=2)
    cfg = oracle.make_cfg(sh_degree=3)
    w = np.random.default_rng(1).standard_normal((2, 24, 32, 3))
    _, _, both, _ = _backward_f64(oracle, cfg, sc, w)
    tot = None
    for k in range(2):
        s1 = dict(sc); s1["cameras"] = [sc["cameras"][k]]
        _, _, g, _ = _backward_f64(oracle, cfg, s1, w[k:k + 1])
        tot = g if tot is None else {n: tot[n] + g[n] for n in g}
    for n in both:
        np.testing.assert_allclose(both[n], tot[n], rtol=1e-11, atol=1e-14)
