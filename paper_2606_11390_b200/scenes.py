"""Seeded synthetic scene generators (inputs only).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path.  It holds none of
the method's arithmetic: it draws Gaussian parameter arrays, builds pinhole cameras with
``look_at`` and draws target images.  Nothing here projects, bins, sorts or composites.

The five recipes follow BASELINE.json ``configs`` as made concrete in SURVEY.md §8(d)
(draw order: means, log_scales, quats, opacity logits, sh_dc, sh_rest, target image).
They stand in for the paper's Mip-NeRF 360 and aerial captures (Table 2,
:205 Fig. 1, :209 Fig. 2), which are not available here.

Cameras are plain dicts with keys ``width, height, fx, fy, cx, cy, near, far, viewmat``
(``viewmat`` = row-major 3x4 world->camera ``[W|tau]``, camera axes +x right, +y down,
+z forward).
"""
from __future__ import annotations

import numpy as np

NEAR_DEFAULT = 0.2          # SURVEY.md §8(c) reading A4
FAR_INF = 3.0e38            # "no far plane" as a finite fp32 value

__all__ = ["make_scene", "look_at", "make_camera", "target_image", "SCENES", "NEAR_DEFAULT", "FAR_INF"]


def look_at(eye, target, up):
    """World->camera matrix per SURVEY.md §8(d): f = normalize(target-eye),
    d = -normalize(up - (up.f) f), r = d x f, W = [r; d; f], tau = -W eye."""
    eye = np.asarray(eye, dtype=np.float64)
    target = np.asarray(target, dtype=np.float64)
    up = np.asarray(up, dtype=np.float64)
    f = target - eye
    f /= np.linalg.norm(f)
    d = up - np.dot(up, f) * f
    d = -d / np.linalg.norm(d)
    r = np.cross(d, f)
    W = np.stack([r, d, f], axis=0)
    tau = -W @ eye
    return np.concatenate([W, tau[:, None]], axis=1)  # 3x4


def make_camera(width, height, fx, fy, eye, target, up, cx=None, cy=None,
                near=NEAR_DEFAULT, far=FAR_INF):
    vm = look_at(eye, target, up)
    return {
        "width": int(width), "height": int(height),
        "fx": float(fx), "fy": float(fy),
        "cx": float(width / 2 if cx is None else cx),
        "cy": float(height / 2 if cy is None else cy),
        "near": float(near), "far": float(far),
        "viewmat": vm.astype(np.float64),
    }


def _normal(rng, shape, mean, std):
    x = rng.standard_normal(shape, dtype=np.float32)
    x *= np.float32(std)
    x += np.float32(mean)
    return x


def _sh(rng, n, deg, dc_std, rest_std):
    K = (deg + 1) ** 2
    sh = np.empty((n, K, 3), dtype=np.float32)
    sh[:, 0, :] = _normal(rng, (n, 3), 0.0, dc_std)
    if K > 1:
        sh[:, 1:, :] = _normal(rng, (n, K - 1, 3), 0.0, rest_std)
    return sh


def _quats(rng, n):
    q = rng.standard_normal((n, 4), dtype=np.float32)
    q /= np.linalg.norm(q, axis=1, keepdims=True).astype(np.float32)
    return q


def _pack(means, log_scales, quats, logits, sh, deg, cams, bg=(0.0, 0.0, 0.0), name=""):
    return {
        "name": name,
        "means": np.ascontiguousarray(means, dtype=np.float32),
        "log_scales": np.ascontiguousarray(log_scales, dtype=np.float32),
        "quats": np.ascontiguousarray(quats, dtype=np.float32),
        "opacity_logits": np.ascontiguousarray(logits, dtype=np.float32),
        "sh": np.ascontiguousarray(sh, dtype=np.float32),
        "sh_degree": int(deg),
        "cameras": cams,
        "bg": np.asarray(bg, dtype=np.float32),
    }


def scene_tiny(n=None, seed=0):
    n = 1024 if n is None else n
    rng = np.random.Generator(np.random.PCG64(seed))
    means = rng.uniform(-1.0, 1.0, (n, 3)).astype(np.float32)
    ls = _normal(rng, (n, 3), -3.0, 0.3)
    q = _quats(rng, n)
    lo = _normal(rng, (n,), 0.0, 1.0)
    sh = _sh(rng, n, 0, 0.5, 0.0)
    cams = [make_camera(64, 64, 64.0, 64.0, (0, 0, -3), (0, 0, 0), (0, -1, 0))]
    return _pack(means, ls, q, lo, sh, 0, cams, name="tiny")


def scene_object(n=None, seed=1, views=8):
    n = 100_000 if n is None else n
    rng = np.random.Generator(np.random.PCG64(seed))
    means = _normal(rng, (n, 3), 0.0, 0.5)
    ls = _normal(rng, (n, 3), -4.5, 0.5)
    q = _quats(rng, n)
    lo = _normal(rng, (n,), 0.0, 1.5)
    sh = _sh(rng, n, 3, 0.5, 0.05)
    cams = []
    for k in range(views):
        th = 2.0 * np.pi * k / 8
        eye = (3.0 * np.sin(th), 0.0, -3.0 * np.cos(th))
        cams.append(make_camera(1920, 1080, 1500.0, 1500.0, eye, (0, 0, 0), (0, -1, 0)))
    return _pack(means, ls, q, lo, sh, 3, cams, name="object")


def scene_room(n=None, seed=2, views=4):
    n = 1_000_000 if n is None else n
    rng = np.random.Generator(np.random.PCG64(seed))
    means = rng.uniform(0.0, 1.0, (n, 3)).astype(np.float32)
    means *= np.array([10.0, 4.0, 10.0], dtype=np.float32)
    ls = _normal(rng, (n, 3), -4.0, 0.6)
    q = _quats(rng, n)
    lo = _normal(rng, (n,), -0.5, 2.0)
    sh = _sh(rng, n, 3, 0.5, 0.05)
    eyes = [(2.5, 1.6, 2.5), (7.5, 1.6, 2.5), (7.5, 1.6, 7.5), (2.5, 1.6, 7.5)][:views]
    cams = [make_camera(3840, 2160, 3000.0, 3000.0, e, (5, 2, 5), (0, 1, 0)) for e in eyes]
    return _pack(means, ls, q, lo, sh, 3, cams, name="room")


def _clustered(rng, n, n_clusters, extent, spacing, hmax, sigma):
    """Cluster centres on a street grid: pick an axis, one of the grid lines, a uniform
    position along it and a uniform height; members = centre + N(0, sigma^2)^3 (z up)."""
    n_lines = int(round(extent / spacing)) + 1
    axis = rng.integers(0, 2, n_clusters)
    line = rng.integers(0, n_lines, n_clusters).astype(np.float64) * spacing
    along = rng.uniform(0.0, extent, n_clusters)
    h = rng.uniform(0.0, hmax, n_clusters)
    cx = np.where(axis == 0, along, line)
    cy = np.where(axis == 0, line, along)
    centres = np.stack([cx, cy, h], axis=1).astype(np.float32)
    member = rng.integers(0, n_clusters, n)
    means = _normal(rng, (n, 3), 0.0, sigma)
    means += centres[member]
    return means


def scene_block(n=None, seed=3):
    n = 10_000_000 if n is None else n
    rng = np.random.Generator(np.random.PCG64(seed))
    means = _clustered(rng, n, 2000, 500.0, 50.0, 40.0, 2.0)
    ls = _normal(rng, (n, 3), -3.0, 0.8)
    q = _quats(rng, n)
    lo = _normal(rng, (n,), -1.0, 2.0)
    sh = _sh(rng, n, 3, 0.5, 0.05)
    cams = [make_camera(3840, 2160, 3000.0, 3000.0, (250, 250, 1.7), (251, 250, 1.7), (0, 0, 1), far=120.0)]
    return _pack(means, ls, q, lo, sh, 3, cams, name="block")


def scene_city(n=None, seed=4, views=4, far=120.0):
    n = 60_000_000 if n is None else n
    rng = np.random.Generator(np.random.PCG64(seed))
    means = _clustered(rng, n, 20000, 2000.0, 100.0, 60.0, 3.0)
    ls = _normal(rng, (n, 3), -3.0, 1.0)
    q = _quats(rng, n)
    lo = _normal(rng, (n,), -1.0, 2.0)
    sh = _sh(rng, n, 3, 0.5, 0.05)
    poses = [((1000, 1000, 1.7), (1, 0, 0)), ((500, 700, 1.7), (0, 1, 0)),
             ((1500, 300, 1.7), (-1, 0, 0)), ((200, 1800, 1.7), (0, -1, 0))][:views]
    cams = []
    for eye, d in poses:
        tgt = (eye[0] + d[0], eye[1] + d[1], eye[2] + d[2])
        cams.append(make_camera(3840, 2160, 3000.0, 3000.0, eye, tgt, (0, 0, 1), far=far))
    return _pack(means, ls, q, lo, sh, 3, cams, name="city")


SCENES = {"tiny": scene_tiny, "object": scene_object, "room": scene_room,
          "block": scene_block, "city": scene_city}


def make_scene(name, n=None, **kw):
    """Build one of the five seeded scenes; ``n`` overrides the Gaussian count (tests use
    reduced counts of the same distribution)."""
    return SCENES[name](n=n, **kw)


def target_image(scene, seed_offset=1000):
    """Seeded uniform[0,1) target images [C,H,W,3] (SURVEY.md §8(c) reading A18)."""
    cams = scene["cameras"]
    seed = {"tiny": 0, "object": 1, "room": 2, "block": 3, "city": 4}.get(scene["name"], 0)
    rng = np.random.Generator(np.random.PCG64(seed + seed_offset))
    return rng.random((len(cams), cams[0]["height"], cams[0]["width"], 3), dtype=np.float32)
