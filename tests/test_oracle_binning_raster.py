"""Pins for the oracle's binning (O-B) and forward compositing (O-R1) stages
(SURVEY.md §8(c); PAPER.md:96 "sorts the Gaussians by depth, rasterizes them", :205
"intersection records").  Brute force on tiny inputs, invariants named in north_star
(transmittance monotone, empty tile -> background, permutation invariance), the textbook
"over" operator and an untiled brute-force renderer.
"""
import struct

import numpy as np
import pytest

from paper_2606_11390_b200 import scenes


def _proj(oracle, sc, cfg, cams=None):
    cams = sc["cameras"] if cams is None else cams
    return oracle.project_fwd(cfg, sc["means"], sc["log_scales"], sc["quats"], sc["opacity_logits"], sc["sh"], cams)


def _f32bits(x):
    return struct.unpack("<I", struct.pack("<f", float(x)))[0]


# ------------------------------------------------------------------ O-B brute force
@pytest.mark.parametrize("scene,n,ncam", [("tiny", None, 1), ("object", 400, 3)])
def test_binning_matches_brute_force(oracle, scene, n, ncam):
    sc = scenes.make_scene(scene, n=n)
    cams = sc["cameras"][:ncam]
    cfg = oracle.make_cfg(sh_degree=sc["sh_degree"])
    pf = _proj(oracle, sc, cfg, cams)
    m2d = pf["means2d"].astype(np.float32)
    dep = pf["depths"].astype(np.float32)
    keys, vals, ranges = oracle.bin_tiles(cfg, cams, m2d, dep, pf["radii"])
    W, H = cams[0]["width"], cams[0]["height"]
    Gx, Gy = (W + 15) // 16, (H + 15) // 16
    N = sc["means"].shape[0]
    # brute force: every (view, Gaussian, tile) triple, overlap decided by interval arithmetic on the
    # fp32 bounds (tile tx covered iff 16tx+16 > u-r and 16tx+16 <= u+r+15)
    recs = []
    for c in range(ncam):
        for i in range(N):
            r = int(pf["radii"][c, i])
            if r == 0:
                continue
            lo = [np.float32(m2d[c, i, a]) - np.float32(r) for a in range(2)]
            hi = [np.float32(m2d[c, i, a]) + np.float32(r + 15) for a in range(2)]
            for ty in range(Gy):
                if not (16 * ty + 16 > lo[1] and 16 * ty + 16 <= hi[1]):
                    continue
                for tx in range(Gx):
                    if 16 * tx + 16 > lo[0] and 16 * tx + 16 <= hi[0]:
                        key = ((c * Gx * Gy + ty * Gx + tx) << 32) | _f32bits(dep[c, i])
                        recs.append((key, c * N + i))
    assert len(recs) == len(keys) == int(pf["tiles_touched"].sum())
    recs.sort(key=lambda kv: kv[0])                      # Python's sort is stable: ties keep (view, index) order
    np.testing.assert_array_equal(keys, np.array([k for k, _ in recs], dtype=np.uint64))
    np.testing.assert_array_equal(vals, np.array([v for _, v in recs], dtype=np.int32))
    # ranges partition [0, M) in tile order; empty tiles are [0, 0) (reading A14)
    M = len(keys)
    tile_of = (keys >> np.uint64(32)).astype(np.int64)
    pos = 0
    for t in range(ncam * Gx * Gy):
        cnt = int((tile_of == t).sum())
        if cnt == 0:
            assert tuple(ranges[t]) == (0, 0)
        else:
            assert tuple(ranges[t]) == (pos, pos + cnt)
            seg_depth = dep.reshape(-1)[vals[pos:pos + cnt]]
            assert np.all(np.diff(seg_depth) >= 0)
            pos += cnt
    assert pos == M


def test_binning_ties_keep_index_order(oracle):
    """Reading A10: equal (tile, depth) keys keep ascending Gaussian index."""
    cfg = oracle.make_cfg(sh_degree=0)
    cam = scenes.make_camera(64, 64, 64.0, 64.0, (0, 0, -3), (0, 0, 0), (0, -1, 0))
    m2d = np.array([[[20.0, 20.0], [21.0, 20.0], [19.0, 22.0], [22.0, 21.0]]], np.float32)
    dep = np.array([[3.0, 2.0, 3.0, 3.0]], np.float32)
    rad = np.array([[2, 2, 2, 2]], np.int32)
    keys, vals, ranges = oracle.bin_tiles(cfg, [cam], m2d, dep, rad)
    t = 1 * 4 + 1
    s, e = ranges[t]
    np.testing.assert_array_equal(vals[s:e], [1, 0, 2, 3])


def test_depth_bits_are_order_preserving():
    d = np.sort(np.random.default_rng(0).uniform(0.2, 500.0, 1000).astype(np.float32))
    bits = d.view(np.uint32).astype(np.int64)
    assert np.all(np.diff(bits) >= 0)


# ------------------------------------------------------------------ O-R1 invariants
def test_empty_tile_gives_background(oracle):
    sc = scenes.make_scene("tiny", n=40)
    sc["bg"] = np.array([0.2, 0.4, 0.6], np.float32)
    cfg = oracle.make_cfg(sh_degree=0)
    r = oracle.render(cfg, sc)
    Gx = 4
    empties = 0
    for t in range(16):
        if r["ranges"][t, 0] == r["ranges"][t, 1]:
            ty, tx = divmod(t, Gx)
            blk = r["image"][0, 16 * ty:16 * ty + 16, 16 * tx:16 * tx + 16]
            np.testing.assert_array_equal(blk, np.broadcast_to(sc["bg"].astype(np.float64), blk.shape))
            np.testing.assert_array_equal(r["final_T"][0, 16 * ty:16 * ty + 16, 16 * tx:16 * tx + 16], 1.0)
            np.testing.assert_array_equal(r["n_contrib"][0, 16 * ty:16 * ty + 16, 16 * tx:16 * tx + 16], 0)
            empties += 1
    assert empties >= 1


def test_transmittance_is_monotone_and_bounded(oracle):
    """Render with the per-tile lists truncated to their first k entries: final_T(k) must be
    non-increasing in k and stay within [t_min, 1]."""
    sc = scenes.make_scene("tiny")
    sc["opacity_logits"] = sc["opacity_logits"] + 2.0          # make pixels saturate
    cfg = oracle.make_cfg(sh_degree=0)
    r = oracle.render(cfg, sc)
    prev = np.ones((1, 64, 64))
    maxlen = int((r["ranges"][:, 1] - r["ranges"][:, 0]).max())
    for k in list(range(0, 40)) + list(range(40, maxlen + 16, 16)):
        rg = r["ranges"].copy()
        rg[:, 1] = np.minimum(rg[:, 1], rg[:, 0] + k)
        _, T, nc = oracle.raster_fwd(cfg, sc["cameras"], r["vals"], rg, r["rec"]["means2d"], r["rec"]["conics"],
                                     r["rec"]["opacities"], r["rec"]["rgbs"], sc["bg"])
        assert np.all(T <= prev + 0.0)
        assert np.all(T >= cfg["t_min"]) and np.all(T <= 1.0)
        assert np.all(nc <= k)
        prev = T
    np.testing.assert_array_equal(prev, r["final_T"])
    assert (r["final_T"] < 0.01).sum() > 100                   # saturation (early termination) is exercised


def test_storage_permutation_with_same_depth_order_leaves_image_unchanged(oracle):
    sc = scenes.make_scene("tiny")
    cfg = oracle.make_cfg(sh_degree=0)
    # drop Gaussians whose fp32 depth collides with another's, so that the depth order is unique
    d = oracle.render(cfg, sc)["rec"]["depths"][0]
    _, first, counts = np.unique(d, return_index=True, return_counts=True)
    keep = np.sort(first[counts == 1])
    assert len(keep) > 900
    for k in ("means", "log_scales", "quats", "opacity_logits", "sh"):
        sc[k] = np.ascontiguousarray(sc[k][keep])
    r0 = oracle.render(cfg, sc)
    d = r0["rec"]["depths"][0]
    assert len(np.unique(d)) == len(d)                         # no depth ties -> order is unique
    perm = np.random.default_rng(7).permutation(len(d))
    sc2 = dict(sc)
    for k in ("means", "log_scales", "quats", "opacity_logits", "sh"):
        sc2[k] = np.ascontiguousarray(sc[k][perm])
    r1 = oracle.render(cfg, sc2)
    np.testing.assert_array_equal(r0["image"], r1["image"])
    np.testing.assert_array_equal(r0["final_T"], r1["final_T"])
    np.testing.assert_array_equal(r0["n_contrib"], r1["n_contrib"])


def test_two_flat_layers_reproduce_over_operator(oracle):
    """Two very wide Gaussians (conic ~ 0, so alpha = opacity everywhere) give the textbook
    'over' compositing c1 a1 + c2 a2 (1 - a1) + (1 - a1)(1 - a2) bg."""
    cfg = oracle.make_cfg(sh_degree=0)
    cam = scenes.make_camera(32, 32, 32.0, 32.0, (0, 0, -3), (0, 0, 0), (0, -1, 0))
    m2d = np.array([[[16.0, 16.0], [16.0, 16.0]]])
    con = np.full((1, 2, 3), 0.0)
    op = np.array([[0.6, 0.3]])
    rgb = np.array([[[1.0, 0.2, 0.1], [0.1, 0.9, 0.5]]])
    bg = np.array([0.05, 0.1, 0.2])
    # entry order: Gaussian 1 in front of Gaussian 0
    vals = np.array([1, 0] * 4, np.int32)
    ranges = np.array([[0, 2], [2, 4], [4, 6], [6, 8]], np.int64)
    img, T, nc = oracle.raster_fwd(cfg, [cam], vals, ranges, m2d, con, op, rgb, bg)
    want = rgb[0, 1] * 0.3 + rgb[0, 0] * 0.6 * 0.7 + 0.7 * 0.4 * bg
    np.testing.assert_allclose(img, np.broadcast_to(want, img.shape), rtol=1e-14)
    np.testing.assert_allclose(T, 0.28, rtol=1e-14)
    assert np.all(nc == 2)


def test_alpha_rules(oracle):
    """Reading A11: alpha clamps at 0.99; alpha < 1/255 is skipped but still counted by the
    running index; compositing stops BEFORE the entry that would take T below 1e-4."""
    cfg = oracle.make_cfg(sh_degree=0)
    cam = scenes.make_camera(16, 16, 16.0, 16.0, (0, 0, -3), (0, 0, 0), (0, -1, 0))
    n = 5
    m2d = np.tile([8.0, 8.0], (1, n, 1))
    con = np.zeros((1, n, 3))
    rgb = np.ones((1, n, 3)) * np.arange(1, n + 1)[None, :, None] * 0.1
    op = np.array([[0.999, 0.003, 0.999, 0.5, 0.5]])        # clamp, skip, clamp, would terminate, never reached
    vals = np.arange(n, dtype=np.int32)
    ranges = np.array([[0, n]], np.int64)
    img, T, nc = oracle.raster_fwd(cfg, [cam], vals, ranges, m2d, con, op, rgb, np.zeros(3))
    # T after entry 0: 0.01; entry 1 skipped (0.003 < 1/255); after entry 2: 1e-4 (not < 1e-4);
    # entry 3: T' = 5e-5 < 1e-4 -> stop, entry 3 not composited
    np.testing.assert_allclose(T, 0.01 * 0.01, rtol=1e-12)
    np.testing.assert_allclose(img[0, 0, 0], 0.1 * 0.99 + 0.3 * 0.99 * 0.01, rtol=1e-12)
    assert np.all(nc == 3)
    # power > 0 is skipped: an indefinite conic makes power positive along the diagonal
    con2 = np.zeros((1, 1, 3)); con2[0, 0] = [0.0, -0.01, 0.0]
    img2, T2, nc2 = oracle.raster_fwd(cfg, [cam], np.array([0], np.int32), np.array([[0, 1]], np.int64),
                                      np.array([[[8.0, 8.0]]]), con2, np.array([[0.5]]), np.ones((1, 1, 3)), np.zeros(3))
    assert T2[0, 0, 0] == 1.0 and nc2[0, 0, 0] == 0          # dx*dy > 0 there -> power = +dx*dy > 0
    assert T2[0, 0, 15] < 1.0                                  # dx*dy < 0 -> contributes


def _untiled_render(cfg, cams, rec, radii, bg):
    """Brute force without tiles: every pixel x every visible Gaussian of the view, sorted by
    (fp32 depth, index), same alpha rules.  Plain numpy, vectorised over pixels."""
    C = len(cams)
    W, H = cams[0]["width"], cams[0]["height"]
    out = np.zeros((C, H, W, 3))
    Tout = np.zeros((C, H, W))
    jj, ii = np.meshgrid(np.arange(W) + 0.5, np.arange(H) + 0.5)
    for c in range(C):
        idx = np.nonzero(radii[c] > 0)[0]
        idx = idx[np.argsort(rec["depths"][c, idx], kind="stable")]
        T = np.ones((H, W)); col = np.zeros((H, W, 3)); alive = np.ones((H, W), bool)
        for g in idx:
            dx = np.float64(rec["means2d"][c, g, 0]) - jj
            dy = np.float64(rec["means2d"][c, g, 1]) - ii
            A, B, Cc = [np.float64(v) for v in rec["conics"][c, g]]
            power = -0.5 * (A * dx * dx + Cc * dy * dy) - B * dx * dy
            alpha = np.minimum(cfg["alpha_max"], np.float64(rec["opacities"][c, g]) * np.exp(power))
            ok = alive & (power <= 0) & (alpha >= cfg["alpha_min"])
            Tn = T * (1 - alpha)
            stop = ok & (Tn < cfg["t_min"])
            alive &= ~stop
            ok &= ~stop
            col += np.where(ok[..., None], (alpha * T)[..., None] * rec["rgbs"][c, g].astype(np.float64), 0.0)
            T = np.where(ok, Tn, T)
        out[c] = col + T[..., None] * np.asarray(bg, np.float64)
        Tout[c] = T
    return out, Tout


def test_tiled_render_equals_untiled_brute_force_when_extent_is_large(oracle):
    sc = scenes.make_scene("object", n=150)
    sc["log_scales"] = sc["log_scales"] + 1.5
    cams = [scenes.make_camera(96, 64, 80.0, 80.0, (0.5, 0.3, -3.0), (0, 0, 0), (0, -1, 0)),
            scenes.make_camera(96, 64, 80.0, 80.0, (-2.0, 0.5, -2.0), (0, 0, 0), (0, -1, 0))]
    sc["cameras"] = cams
    sc["bg"] = np.array([0.1, 0.2, 0.3], np.float32)
    cfg = oracle.make_cfg(extent=200.0)                        # every visible Gaussian reaches every tile
    r = oracle.render(cfg, sc)
    assert np.all(r["proj"]["tiles_touched"][r["proj"]["radii"] > 0] == 6 * 4)
    img, T = _untiled_render(cfg, cams, r["rec"], r["proj"]["radii"], sc["bg"])
    np.testing.assert_allclose(r["image"], img, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(r["final_T"], T, rtol=1e-12, atol=1e-14)
    # with the default 3-sigma extent the difference is bounded by the truncated tails
    r3 = oracle.render(oracle.make_cfg(), sc)
    assert np.abs(r3["image"] - img).max() < 0.08
    assert np.abs(r3["image"] - img).mean() < 2e-3


def test_batched_views_equal_single_view_runs(oracle):
    sc = scenes.make_scene("object", n=500)
    cams = [scenes.make_camera(128, 96, 100.0, 100.0, e, (0, 0, 0), (0, -1, 0)) for e in [(0, 0, -3), (3, 0, 0), (0.5, 2, -2)]]
    sc["cameras"] = cams
    cfg = oracle.make_cfg()
    r = oracle.render(cfg, sc)
    for k, cam in enumerate(cams):
        s1 = dict(sc); s1["cameras"] = [cam]
        r1 = oracle.render(cfg, s1)
        np.testing.assert_array_equal(r["image"][k], r1["image"][0])
        np.testing.assert_array_equal(r["n_contrib"][k], r1["n_contrib"][0])


def test_float_oracle_sits_at_fp32_noise_floor(oracle):
    sc = scenes.make_scene("tiny")
    cfg = oracle.make_cfg(sh_degree=0)
    r64 = oracle.render(cfg, sc, np.float64)
    r32 = oracle.render(cfg, sc, np.float32)
    assert np.abs(r64["image"] - r32["image"]).max() < 1e-5
