"""Pins for the oracle's per-Gaussian forward stage O-P1.

Each test checks the oracle against something other than itself: a closed form, a library
routine (scipy rotations, scipy spherical harmonics, numpy eigen-solver), a numerical
Jacobian / Monte-Carlo estimate of the definition, or exact integer reasoning.
"""
import json
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy.spatial.transform import Rotation
from scipy.special import expit, sph_harm_y

from paper_2606_11390_b200 import scenes

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _cam(width=64, height=64, f=64.0, eye=(0, 0, -3), target=(0, 0, 0), up=(0, -1, 0), **kw):
    return scenes.make_camera(width, height, f, f, eye, target, up, **kw)


def _one(oracle, cfg, mean, ls, q, logit, sh, cams):
    K = (cfg["sh_degree"] + 1) ** 2
    sh = np.zeros((1, K, 3)) if sh is None else np.asarray(sh, dtype=np.float64).reshape(1, K, 3)
    return oracle.project_fwd(cfg, np.asarray([mean], float), np.asarray([ls], float), np.asarray([q], float),
                              np.asarray([logit], float), sh, cams)


# ------------------------------------------------------------------ covariance (step 2)
def test_cov3d_matches_library_rotation(oracle):
    rng = np.random.default_rng(0)
    for _ in range(50):
        q = rng.standard_normal(4) * rng.uniform(0.2, 3.0)      # unnormalised on purpose (reading A1)
        ls = rng.normal(-2, 1, 3)
        S = oracle.cov3d(ls, q)
        R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()   # scipy is (x,y,z,w); ours (w,x,y,z) (A2)
        want = R @ np.diag(np.exp(2 * ls)) @ R.T
        np.testing.assert_allclose(S, want, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(S, S.T, atol=0)
        np.testing.assert_allclose(np.sort(np.linalg.eigvalsh(S)), np.sort(np.exp(2 * ls)), rtol=1e-10)


def test_cov3d_special_cases(oracle):
    ls = np.log([0.5, 2.0, 3.0])
    np.testing.assert_allclose(oracle.cov3d(ls, [1, 0, 0, 0]), np.diag([0.25, 4.0, 9.0]), rtol=1e-14)
    # 90 degrees about z swaps the x and y variances
    q = [np.cos(np.pi / 4), 0, 0, np.sin(np.pi / 4)]
    np.testing.assert_allclose(oracle.cov3d(ls, q), np.diag([4.0, 0.25, 9.0]), rtol=1e-12, atol=1e-14)
    # 90 degrees about x maps +y to +z (right-handed): variances (x, z, y)
    q = [np.cos(np.pi / 4), np.sin(np.pi / 4), 0, 0]
    np.testing.assert_allclose(oracle.cov3d(ls, q), np.diag([0.25, 9.0, 4.0]), rtol=1e-12, atol=1e-14)


def test_rotation_handedness_off_diagonal(oracle):
    # a small positive rotation about z tilts the long x axis towards +y: Sigma_xy > 0
    th = 0.3
    S = oracle.cov3d(np.log([2.0, 0.1, 0.1]), [np.cos(th / 2), 0, 0, np.sin(th / 2)])
    assert S[0, 1] > 0
    np.testing.assert_allclose(S[0, 1], (4.0 - 0.01) * np.sin(th) * np.cos(th), rtol=1e-12)


# ------------------------------------------------------------------ spherical harmonics (step 9)
def _library_real_sh(l, m, d):
    """Real SH with Condon-Shortley phase from scipy's complex Y_l^m."""
    theta = np.arccos(np.clip(d[2], -1, 1))
    phi = np.arctan2(d[1], d[0])
    if m == 0:
        return sph_harm_y(l, 0, theta, phi).real
    y = sph_harm_y(l, abs(m), theta, phi)
    return np.sqrt(2.0) * (y.real if m > 0 else y.imag)


def test_sh_basis_matches_library(oracle):
    rng = np.random.default_rng(1)
    for _ in range(40):
        d = rng.standard_normal(3)
        d /= np.linalg.norm(d)
        Y = oracle.sh_basis(d)
        k = 0
        for l in range(4):
            for m in range(-l, l + 1):
                np.testing.assert_allclose(Y[k], _library_real_sh(l, m, d), rtol=1e-10, atol=1e-12, err_msg=f"l={l} m={m}")
                k += 1


def test_sh_basis_orthonormal_by_quadrature(oracle):
    xs, ws = np.polynomial.legendre.leggauss(12)
    nphi = 24
    G = np.zeros((16, 16))
    for ct, w in zip(xs, ws):
        st = np.sqrt(1 - ct * ct)
        for j in range(nphi):
            ph = 2 * np.pi * (j + 0.5) / nphi
            Y = oracle.sh_basis([st * np.cos(ph), st * np.sin(ph), ct])
            G += w * (2 * np.pi / nphi) * np.outer(Y, Y)
    np.testing.assert_allclose(G, np.eye(16), atol=1e-12)


def test_sh_constants_golden(oracle):
    g = json.load(open(os.path.join(GOLD, "sh_constants.json")))
    np.testing.assert_allclose(oracle.sh_basis([0, 0, 1])[0], g["c0"], rtol=1e-15)
    np.testing.assert_allclose(oracle.sh_basis([0, 0, 1])[2], g["c1"], rtol=1e-15)
    np.testing.assert_allclose(oracle.sh_basis([0, 0, 1])[6], 2 * g["c2b"], rtol=1e-15)
    np.testing.assert_allclose(oracle.sh_basis([0, 0, 1])[12], 2 * g["c3d"], rtol=1e-15)
    s = np.sqrt(0.5)
    np.testing.assert_allclose(oracle.sh_basis([s, s, 0])[4], g["c2a"] * 0.5, rtol=1e-14)
    np.testing.assert_allclose(oracle.sh_basis([1, 0, 0])[8], g["c2c"], rtol=1e-15)
    np.testing.assert_allclose(oracle.sh_basis([1, 0, 0])[15], -g["c3a"], rtol=1e-15)
    t = 1 / np.sqrt(3.0)
    np.testing.assert_allclose(oracle.sh_basis([t, t, t])[10], g["c3b"] * t ** 3, rtol=1e-14)
    np.testing.assert_allclose(oracle.sh_basis([0, s, s])[11], -g["c3c"] * s * (4 * 0.5 - 0.5), rtol=1e-14)
    np.testing.assert_allclose(oracle.sh_basis([s, 0, s])[14], g["c3e"] * s * 0.5, rtol=1e-14)


def test_sh_degree0_colour_is_constant(oracle):
    """north_star: "SH degree 0 gives the constant C0*f_dc+0.5"."""
    g = json.load(open(os.path.join(GOLD, "sh_constants.json")))
    cfg = oracle.make_cfg(sh_degree=0)
    f = np.array([0.3, -0.7, 1.1])
    for eye in [(0, 0, -3), (2, 1, -2), (-1, 2, 3)]:
        out = _one(oracle, cfg, (0.1, 0.05, 0.0), (-3, -3, -3), (1, 0, 0, 0), 0.0, f, [_cam(eye=eye)])
        assert out["radii"][0, 0] > 0
        np.testing.assert_allclose(out["rgbs"][0, 0], g["c0"] * f + 0.5, rtol=1e-14)
    # the clamp at zero (reading A15)
    out = _one(oracle, cfg, (0, 0, 0), (-3, -3, -3), (1, 0, 0, 0), 0.0, [-5.0, 0.0, 5.0], [_cam()])
    np.testing.assert_allclose(out["rgbs"][0, 0], [0.0, 0.5, g["c0"] * 5 + 0.5], rtol=1e-14)


def test_sh_colour_uses_camera_to_gaussian_direction(oracle):
    # degree 1, coefficient only on Y_2 (= c1 z): colour = c1 * dir_z * f + 0.5 with dir from camera to Gaussian
    cfg = oracle.make_cfg(sh_degree=1)
    sh = np.zeros((4, 3))
    sh[2] = 1.0
    eye = np.array([1.0, -2.0, -3.0])
    p = np.array([0.2, 0.1, 0.4])
    out = _one(oracle, cfg, p, (-3, -3, -3), (1, 0, 0, 0), 0.0, sh, [_cam(eye=eye, target=p)])
    d = (p - eye) / np.linalg.norm(p - eye)
    np.testing.assert_allclose(out["rgbs"][0, 0], np.sqrt(3 / (4 * np.pi)) * d[2] + 0.5, rtol=1e-12)


# ------------------------------------------------------------------ projection (steps 1, 3-7)
def _pinhole(cam, p):
    vm = np.asarray(cam["viewmat"])
    t = vm[:, :3] @ p + vm[:, 3]
    return np.array([cam["fx"] * t[0] / t[2] + cam["cx"], cam["fy"] * t[1] / t[2] + cam["cy"]]), t


def test_mean2d_depth_match_pinhole_definition(oracle):
    rng = np.random.default_rng(2)
    cfg = oracle.make_cfg(sh_degree=0)
    cam = _cam(640, 480, 500.0, eye=(1.0, -0.5, -4.0), target=(0.2, 0.1, 0.3), up=(0.1, -1, 0.05), cx=300.0, cy=250.0)
    for _ in range(20):
        p = rng.uniform(-1, 1, 3)
        out = _one(oracle, cfg, p, (-3, -3.5, -2.5), rng.standard_normal(4), 0.3, None, [cam])
        uv, t = _pinhole(cam, p)
        np.testing.assert_allclose(out["means2d"][0, 0], uv, rtol=1e-13)
        np.testing.assert_allclose(out["depths"][0, 0], t[2], rtol=1e-13)
        np.testing.assert_allclose(out["opacities"][0, 0], expit(0.3), rtol=1e-14)


def test_ewa_covariance_matches_numerical_jacobian(oracle):
    """Sigma' = J_num (W Sigma W^T) J_num^T with J_num the central-difference Jacobian of the
    pinhole map in camera space; dilation switched off so the conic inverts to Sigma'."""
    rng = np.random.default_rng(3)
    cfg = oracle.make_cfg(sh_degree=0, dilation=0.0)
    cam = _cam(640, 480, 500.0, eye=(1.0, -0.5, -4.0), target=(0.2, 0.1, 0.3), up=(0.1, -1, 0.05))
    vm = np.asarray(cam["viewmat"])
    Wm = vm[:, :3]
    for _ in range(20):
        p = rng.uniform(-1, 1, 3)
        ls = rng.normal(-2.5, 0.5, 3)
        q = rng.standard_normal(4)
        out = _one(oracle, cfg, p, ls, q, 0.0, None, [cam])
        A, B, Cc = out["conics"][0, 0]
        S2 = np.linalg.inv(np.array([[A, B], [B, Cc]]))
        t = Wm @ p + vm[:, 3]
        f = lambda tt: np.array([cam["fx"] * tt[0] / tt[2], cam["fy"] * tt[1] / tt[2]])
        h = 1e-6
        J = np.stack([(f(t + h * e) - f(t - h * e)) / (2 * h) for e in np.eye(3)], axis=1)
        R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()
        Sig = R @ np.diag(np.exp(2 * ls)) @ R.T
        want = J @ Wm @ Sig @ Wm.T @ J.T
        np.testing.assert_allclose(S2, want, rtol=2e-7)


def test_ewa_covariance_monte_carlo(oracle):
    """Sample N(p, Sigma) with small sigma, project every sample exactly, compare the sample
    covariance with Sigma' (first-order agreement)."""
    rng = np.random.default_rng(4)
    cfg = oracle.make_cfg(sh_degree=0, dilation=0.0)
    cam = _cam(640, 480, 500.0, eye=(0.5, 0.2, -4.0), target=(0, 0, 0), up=(0, -1, 0))
    p = np.array([0.4, -0.3, 0.5])
    ls = np.log([0.010, 0.004, 0.007])
    q = np.array([0.9, 0.2, -0.3, 0.1])
    out = _one(oracle, cfg, p, ls, q, 0.0, None, [cam])
    A, B, Cc = out["conics"][0, 0]
    S2 = np.linalg.inv(np.array([[A, B], [B, Cc]]))
    R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()
    L = R @ np.diag(np.exp(ls))
    x = p + rng.standard_normal((400000, 3)) @ L.T
    vm = np.asarray(cam["viewmat"])
    t = x @ vm[:, :3].T + vm[:, 3]
    uv = np.stack([cam["fx"] * t[:, 0] / t[:, 2], cam["fy"] * t[:, 1] / t[:, 2]], axis=1)
    np.testing.assert_allclose(np.cov(uv.T), S2, rtol=2e-2)


def test_dilation_added_to_diagonal_only(oracle):
    cam = _cam(640, 480, 500.0, eye=(0.5, 0.2, -4.0))
    args = ((0.3, 0.1, 0.2), (-2.5, -3.0, -2.0), (0.9, 0.2, -0.3, 0.1), 0.0, None, [cam])
    c0 = _one(oracle, oracle.make_cfg(sh_degree=0, dilation=0.0), *args)["conics"][0, 0]
    c1 = _one(oracle, oracle.make_cfg(sh_degree=0, dilation=0.3), *args)["conics"][0, 0]
    S0 = np.linalg.inv(np.array([[c0[0], c0[1]], [c0[1], c0[2]]]))
    S1 = np.linalg.inv(np.array([[c1[0], c1[1]], [c1[1], c1[2]]]))
    np.testing.assert_allclose(S1 - S0, 0.3 * np.eye(2), atol=1e-9)


def test_jacobian_clamp_limits_off_axis_covariance(oracle):
    """Step 3: beyond 1.3x the half field of view the x/z ratio used in J is frozen, so moving the
    Gaussian further sideways at fixed depth no longer changes Sigma' (mean2d keeps moving)."""
    cfg = oracle.make_cfg(sh_degree=0, dilation=0.0)
    cam = _cam(64, 64, 64.0)            # lim = 1.3 * 64 / 128 = 0.65; depth 3 -> clamp beyond |x| = 1.95
    base = dict(ls=(0.0, 0.0, 0.0), q=(1, 0, 0, 0))     # sigma 1: radius 64 px, still overlaps the image
    c_a = _one(oracle, cfg, (2.5, 0, 0), base["ls"], base["q"], 0.0, None, [cam])
    c_b = _one(oracle, cfg, (3.5, 0, 0), base["ls"], base["q"], 0.0, None, [cam])
    np.testing.assert_allclose(c_a["conics"][0, 0], c_b["conics"][0, 0], rtol=1e-13)
    assert c_b["means2d"][0, 0, 0] > c_a["means2d"][0, 0, 0]
    # and the frozen value is the one at the limit
    c_l = _one(oracle, cfg, (0.65 * 3, 0, 0), base["ls"], base["q"], 0.0, None, [cam])
    np.testing.assert_allclose(c_a["conics"][0, 0], c_l["conics"][0, 0], rtol=1e-12)


def test_radius_matches_library_eigenvalue(oracle):
    rng = np.random.default_rng(5)
    cfg = oracle.make_cfg(sh_degree=0)
    cam = _cam(640, 480, 500.0, eye=(0.5, 0.2, -4.0))
    n = 0
    for _ in range(60):
        out = _one(oracle, cfg, rng.uniform(-1, 1, 3), rng.normal(-2.5, 0.7, 3), rng.standard_normal(4), 0.0, None, [cam])
        if out["radii"][0, 0] == 0:
            continue
        A, B, Cc = out["conics"][0, 0]
        S2 = np.linalg.inv(np.array([[A, B], [B, Cc]]))
        lam = np.linalg.eigvalsh(S2)[-1]
        m = 0.5 * (S2[0, 0] + S2[1, 1])
        if m * m - np.linalg.det(S2) < 0.1:          # eigenvalue floor of reading A6 active
            continue
        np.testing.assert_allclose(out["radius_real"][0, 0], 3.0 * np.sqrt(lam), rtol=1e-9)
        assert out["radii"][0, 0] == int(np.ceil(3.0 * np.sqrt(lam)))
        n += 1
    assert n > 20


def test_near_far_and_offscreen_cull(oracle):
    cfg = oracle.make_cfg(sh_degree=0)
    cam = _cam(near=0.2, far=10.0)       # eye z=-3 looking +z
    vis = lambda p: _one(oracle, cfg, p, (-3, -3, -3), (1, 0, 0, 0), 0.0, None, [cam])
    assert vis((0, 0, 0))["radii"][0, 0] > 0
    for p in [(0, 0, -2.9), (0, 0, -3.0), (0, 0, -5.0), (0, 0, 7.0), (0, 0, 8.0)]:    # tz <= near or >= far
        o = vis(p)
        assert o["radii"][0, 0] == 0 and o["tiles_touched"][0, 0] == 0
    assert vis((0, 0, 6.9))["radii"][0, 0] > 0
    o = vis((30.0, 0, 0))                # far outside the image: no tile overlapped (reading A5)
    assert o["radii"][0, 0] == 0 and o["tiles_touched"][0, 0] == 0


def test_tiles_touched_counts_overlapped_tiles_exactly(oracle):
    """Step 8 re-derived with exact rational arithmetic: tile tx is covered iff
    16 tx + 16 > u - r and 16 tx + 1 <= u + r (the integer meaning of the two floors)."""
    sc = scenes.make_scene("tiny")
    cfg = oracle.make_cfg(sh_degree=0)
    out = oracle.project_fwd(cfg, sc["means"], sc["log_scales"], sc["quats"], sc["opacity_logits"], sc["sh"], sc["cameras"])
    u32 = out["means2d"].astype(np.float32)
    n_checked = 0
    for i in range(sc["means"].shape[0]):
        r = int(out["radii"][0, i])
        if r == 0:
            continue
        cnt = []
        for ax in range(2):
            # the two bounds are evaluated in fp32 (reading A8), then compared exactly
            lo = Fraction(float(np.float32(u32[0, i, ax]) - np.float32(r)))
            hi = Fraction(float(np.float32(u32[0, i, ax]) + np.float32(r + 15)))
            cnt.append(sum(1 for t in range(4) if 16 * t + 16 > lo and 16 * t + 16 <= hi))
        assert out["tiles_touched"][0, i] == cnt[0] * cnt[1]
        n_checked += 1
    assert n_checked > 900


# ------------------------------------------------------------------ closed form (P1 + B + R1)
def test_isotropic_gaussian_closed_form_golden(oracle):
    """north_star: "a single isotropic Gaussian facing the camera renders the analytic
    exp(-r^2/2) falloff times opacity".  Values from tests/golden."""
    g = json.load(open(os.path.join(GOLD, "isotropic_closed_form.json")))
    cfg = oracle.make_cfg(sh_degree=0)
    # principal point at (32, 32.5): the pixel row i=32 (py = 32.5) passes through the centre
    cam = _cam(64, 64, g["fx"], eye=(0, 0, -g["z"]), cx=32.0, cy=32.5)
    logit = np.log(g["opacity"] / (1 - g["opacity"]))
    c0 = 0.28209479177387814
    rgb = np.array([0.9, 0.5, 0.2])
    f_dc = (rgb - 0.5) / c0
    sc = {"means": np.zeros((1, 3)), "log_scales": np.full((1, 3), np.log(g["sigma"])),
          "quats": np.array([[0.3, -0.5, 0.1, 0.8]]),          # isotropic: any rotation
          "opacity_logits": np.array([logit]), "sh": f_dc.reshape(1, 1, 3), "cameras": [cam], "bg": np.zeros(3)}
    r = oracle.render(cfg, sc)
    assert r["proj"]["radii"][0, 0] == g["radius"]
    A, B, Cc = r["proj"]["conics"][0, 0]
    np.testing.assert_allclose([1 / A, 1 / Cc], g["variance"], atol=5e-5)
    assert abs(B) < 1e-12
    for rs, a in g["alpha_at_r"].items():
        j = 32 + int(float(rs) - 0.5)                       # px = j + 0.5 = 32 + r
        for jj in (j, 63 - j):                              # both sides (symmetry)
            np.testing.assert_allclose(r["image"][0, 32, jj], a * rgb, atol=g["abs_tol"])
            np.testing.assert_allclose(r["final_T"][0, 32, jj], 1 - a, atol=g["abs_tol"])
    # full analytic falloff on every pixel: alpha >= 1/255 inside the tile footprint, background elsewhere
    var = (g["fx"] * g["sigma"] / g["z"]) ** 2 + 0.3
    jj, ii = np.meshgrid(np.arange(64) + 0.5, np.arange(64) + 0.5)
    alpha = g["opacity"] * np.exp(-((jj - 32.0) ** 2 + (ii - 32.5) ** 2) / (2 * var))
    alpha[alpha < 1 / 255] = 0
    # footprint: tiles overlapped by the 3-sigma square; here radius 4 around (32, 32.5) touches tiles 1..2 in x and y
    foot = np.zeros((64, 64), bool)
    foot[16:48, 16:48] = True
    np.testing.assert_allclose(r["image"][0], (alpha * foot)[..., None] * rgb, atol=1e-7)
    assert r["proj"]["tiles_touched"][0, 0] == 4


def test_project_is_per_camera_independent(oracle):
    """Batch of cameras = the same Gaussians projected camera by camera."""
    sc = scenes.make_scene("object", n=300)
    cfg = oracle.make_cfg()
    allc = oracle.project_fwd(cfg, sc["means"], sc["log_scales"], sc["quats"], sc["opacity_logits"], sc["sh"], sc["cameras"][:3])
    for k in range(3):
        one = oracle.project_fwd(cfg, sc["means"], sc["log_scales"], sc["quats"], sc["opacity_logits"], sc["sh"], [sc["cameras"][k]])
        for name in ("means2d", "depths", "conics", "opacities", "rgbs", "radii", "tiles_touched"):
            np.testing.assert_array_equal(allc[name][k], one[name][0])
