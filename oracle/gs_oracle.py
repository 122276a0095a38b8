"""ctypes front-end of the CPU oracle (``oracle/gs_oracle.cpp``) -- TEST INFRASTRUCTURE ONLY.

Argument marshalling only: every number is computed in the C++ oracle.  ``dtype`` selects
the ``double`` (truth, finite differences) or ``float`` (fp32 noise floor, timed CPU
baseline) instantiation.  Passages followed: PAPER.md:96, :98 (operators and their
partition axes); SURVEY.md §8(c) O-P1 / O-B / O-R1 / O-R2 / O-P5 (the mathematics).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_LIB = None

DEFAULT_CFG = dict(dilation=0.3, alpha_min=1.0 / 255.0, alpha_max=0.99, t_min=1e-4, extent=3.0,
                   tile=16, sh_degree=3)


def lib():
    global _LIB
    if _LIB is None:
        _LIB = C.CDLL(_build.build())
        _LIB.oracle_bin_tiles.restype = C.c_int64
    return _LIB


def make_cfg(**kw):
    cfg = dict(DEFAULT_CFG)
    cfg.update(kw)
    return cfg


def smooth_cfg(**kw):
    """Thresholds off, so that the rendered image is a differentiable function of the
    parameters (used for finite differences; SURVEY.md §8(c) pins for R2/P5)."""
    cfg = make_cfg(alpha_min=0.0, alpha_max=1.0, t_min=0.0, extent=1.0e4)
    cfg.update(kw)
    return cfg


def _cfg_arr(cfg):
    return np.array([cfg["dilation"], cfg["alpha_min"], cfg["alpha_max"], cfg["t_min"], cfg["extent"],
                     cfg["tile"], cfg["sh_degree"]], dtype=np.float64)


def _cams_arr(cams):
    out = np.zeros((len(cams), 20), dtype=np.float64)
    for k, c in enumerate(cams):
        out[k, :8] = [c["width"], c["height"], c["fx"], c["fy"], c["cx"], c["cy"], c["near"], c["far"]]
        out[k, 8:] = np.asarray(c["viewmat"], dtype=np.float64).reshape(12)
    return out


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _mask(tile_mask):
    """Optional uint8 [C*tiles] selection of tiles to evaluate (sampled checks at full size)."""
    if tile_mask is None:
        return None
    m = np.ascontiguousarray(tile_mask, dtype=np.uint8)
    _mask.keep = m
    return _p(m)


def _suffix(dtype):
    dtype = np.dtype(dtype)
    if dtype == np.float64:
        return "f64"
    if dtype == np.float32:
        return "f32"
    raise ValueError(dtype)


def _as(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def grid(cfg, cam):
    t = int(cfg["tile"])
    return (cam["width"] + t - 1) // t, (cam["height"] + t - 1) // t


def project_fwd(cfg, means, log_scales, quats, opacity_logits, sh, cams, dtype=np.float64):
    """O-P1.  Returns dict of [C,N,*] arrays (+ ``radius_real`` = extent*sqrt(lambda) before ceil)."""
    N = means.shape[0]
    nc = len(cams)
    K = (int(cfg["sh_degree"]) + 1) ** 2
    assert sh.shape == (N, K, 3), (sh.shape, K)
    means, log_scales, quats = _as(means, dtype), _as(log_scales, dtype), _as(quats, dtype)
    opacity_logits, sh = _as(opacity_logits, dtype), _as(sh, dtype)
    out = {
        "means2d": np.zeros((nc, N, 2), dtype), "depths": np.zeros((nc, N), dtype),
        "conics": np.zeros((nc, N, 3), dtype), "opacities": np.zeros((nc, N), dtype),
        "rgbs": np.zeros((nc, N, 3), dtype), "radii": np.zeros((nc, N), np.int32),
        "tiles_touched": np.zeros((nc, N), np.uint32), "radius_real": np.zeros((nc, N), dtype),
    }
    ca, ka = _cfg_arr(cfg), _cams_arr(cams)
    fn = getattr(lib(), "oracle_project_fwd_" + _suffix(dtype))
    fn(_p(ca), C.c_int64(N), _p(means), _p(log_scales), _p(quats), _p(opacity_logits), _p(sh), C.c_int(nc),
       _p(ka), _p(out["means2d"]), _p(out["depths"]), _p(out["conics"]), _p(out["opacities"]), _p(out["rgbs"]),
       _p(out["radii"]), _p(out["tiles_touched"]), _p(out["radius_real"]))
    return out


def bin_tiles(cfg, cams, means2d, depths, radii):
    """O-B for a batch of views.  Inputs are the fp32 means2d/depths and int32 radii, [C,N,*].
    Returns (keys u64[M], vals i32[M], ranges i64[C*tiles,2])."""
    nc = len(cams)
    means2d, depths, radii = _as(means2d, np.float32), _as(depths, np.float32), _as(radii, np.int32)
    N = depths.shape[1]
    assert means2d.shape == (nc, N, 2) and radii.shape == (nc, N)
    W, H = cams[0]["width"], cams[0]["height"]
    gx, gy = grid(cfg, cams[0])
    ca = _cfg_arr(cfg)
    fn = lib().oracle_bin_tiles
    M = fn(_p(ca), C.c_int64(N), C.c_int(nc), C.c_int(W), C.c_int(H), _p(means2d), _p(depths), _p(radii),
           None, None, None)
    keys = np.zeros(M, np.uint64)
    vals = np.zeros(M, np.int32)
    ranges = np.zeros((nc * gx * gy, 2), np.int64)
    M2 = fn(_p(ca), C.c_int64(N), C.c_int(nc), C.c_int(W), C.c_int(H), _p(means2d), _p(depths), _p(radii),
            _p(keys), _p(vals), _p(ranges))
    assert M2 == M
    return keys, vals, ranges


def raster_fwd(cfg, cams, vals, ranges, means2d, conics, opacities, rgbs, bg, dtype=np.float64,
               ambiguity_eps=None, tile_mask=None):
    """O-R1.  Returns (image [C,H,W,3], final_T [C,H,W], n_contrib [C,H,W] i32[, ambiguous u8])."""
    nc = len(cams)
    W, H = cams[0]["width"], cams[0]["height"]
    vals, ranges = _as(vals, np.int32), _as(ranges, np.int64)
    means2d, conics = _as(means2d, dtype), _as(conics, dtype)
    opacities, rgbs, bg = _as(opacities, dtype), _as(rgbs, dtype), _as(bg, dtype)
    image = np.zeros((nc, H, W, 3), dtype)
    final_T = np.zeros((nc, H, W), dtype)
    n_contrib = np.zeros((nc, H, W), np.int32)
    amb = np.zeros((nc, H, W), np.uint8) if ambiguity_eps is not None else None
    ca = _cfg_arr(cfg)
    fn = getattr(lib(), "oracle_raster_fwd_" + _suffix(dtype))
    fn(_p(ca), C.c_int(nc), C.c_int(W), C.c_int(H), _p(vals), _p(ranges), _p(means2d), _p(conics), _p(opacities),
       _p(rgbs), _p(bg), _p(image), _p(final_T), _p(n_contrib), _p(amb) if amb is not None else None,
       C.c_double(0.0 if ambiguity_eps is None else ambiguity_eps), _mask(tile_mask))
    if amb is not None:
        return image, final_T, n_contrib, amb
    return image, final_T, n_contrib


def raster_bwd(cfg, cams, vals, ranges, means2d, conics, opacities, rgbs, bg, final_T, n_contrib, dL_dimage,
               dtype=np.float64, tile_mask=None):
    """O-R2.  Returns dict of per-(view,Gaussian) 2-D gradients shaped like the inputs."""
    nc = len(cams)
    W, H = cams[0]["width"], cams[0]["height"]
    vals, ranges = _as(vals, np.int32), _as(ranges, np.int64)
    means2d, conics = _as(means2d, dtype), _as(conics, dtype)
    opacities, rgbs, bg = _as(opacities, dtype), _as(rgbs, dtype), _as(bg, dtype)
    final_T, n_contrib, dL_dimage = _as(final_T, dtype), _as(n_contrib, np.int32), _as(dL_dimage, dtype)
    ntot = opacities.size
    out = {"means2d": np.zeros(means2d.shape, dtype), "conics": np.zeros(conics.shape, dtype),
           "opacities": np.zeros(opacities.shape, dtype), "rgbs": np.zeros(rgbs.shape, dtype)}
    ca = _cfg_arr(cfg)
    fn = getattr(lib(), "oracle_raster_bwd_" + _suffix(dtype))
    fn(_p(ca), C.c_int(nc), C.c_int(W), C.c_int(H), C.c_int64(ntot), _p(vals), _p(ranges), _p(means2d), _p(conics),
       _p(opacities), _p(rgbs), _p(bg), _p(final_T), _p(n_contrib), _p(dL_dimage), _p(out["means2d"]),
       _p(out["conics"]), _p(out["opacities"]), _p(out["rgbs"]), _mask(tile_mask))
    return out


def project_bwd(cfg, means, log_scales, quats, opacity_logits, sh, cams, radii, g_means2d, g_conics,
                g_opacities, g_rgbs, dtype=np.float64, accumulate_into=None):
    """O-P5.  Returns dict of parameter gradients (means, log_scales, quats, opacity_logits, sh)."""
    N = means.shape[0]
    nc = len(cams)
    means, log_scales, quats = _as(means, dtype), _as(log_scales, dtype), _as(quats, dtype)
    opacity_logits, sh = _as(opacity_logits, dtype), _as(sh, dtype)
    radii = _as(radii, np.int32)
    g_means2d, g_conics = _as(g_means2d, dtype), _as(g_conics, dtype)
    g_opacities, g_rgbs = _as(g_opacities, dtype), _as(g_rgbs, dtype)
    if accumulate_into is None:
        out = {"means": np.zeros((N, 3), dtype), "log_scales": np.zeros((N, 3), dtype),
               "quats": np.zeros((N, 4), dtype), "opacity_logits": np.zeros((N,), dtype),
               "sh": np.zeros(sh.shape, dtype)}
        acc = 0
    else:
        out, acc = accumulate_into, 1
    ca, ka = _cfg_arr(cfg), _cams_arr(cams)
    fn = getattr(lib(), "oracle_project_bwd_" + _suffix(dtype))
    fn(_p(ca), C.c_int64(N), _p(means), _p(log_scales), _p(quats), _p(opacity_logits), _p(sh), C.c_int(nc), _p(ka),
       _p(radii), _p(g_means2d), _p(g_conics), _p(g_opacities), _p(g_rgbs), _p(out["means"]), _p(out["log_scales"]),
       _p(out["quats"]), _p(out["opacity_logits"]), _p(out["sh"]), C.c_int(acc))
    return out


def sh_basis(d, dtype=np.float64):
    d = np.asarray(d, dtype=np.float64)
    Y = np.zeros(16, dtype)
    ct = C.c_double if np.dtype(dtype) == np.float64 else C.c_float
    fn = getattr(lib(), "oracle_sh_basis_" + _suffix(dtype))
    fn.argtypes = [ct, ct, ct, C.c_void_p]
    fn(ct(d[0]), ct(d[1]), ct(d[2]), _p(Y))
    return Y


def cov3d(log_scale, quat, dtype=np.float64):
    ls, q = _as(log_scale, dtype), _as(quat, dtype)
    S = np.zeros((3, 3), dtype)
    getattr(lib(), "oracle_cov3d_" + _suffix(dtype))(_p(ls), _p(q), _p(S))
    return S


def render(cfg, scene, dtype=np.float64, ambiguity_eps=None):
    """Whole forward pass (P1 -> B -> R1) on a scene dict from the shared input generators.
    Stage outputs are handed on exactly as the C-ABI stores them: projected records rounded
    to fp32 (then widened to ``dtype`` again)."""
    cams = scene["cameras"]
    pf = project_fwd(cfg, scene["means"], scene["log_scales"], scene["quats"], scene["opacity_logits"],
                     scene["sh"], cams, dtype)
    rec = {k: pf[k].astype(np.float32) for k in ("means2d", "depths", "conics", "opacities", "rgbs")}
    keys, vals, ranges = bin_tiles(cfg, cams, rec["means2d"], rec["depths"], pf["radii"])
    rf = raster_fwd(cfg, cams, vals, ranges, rec["means2d"], rec["conics"], rec["opacities"], rec["rgbs"],
                    scene["bg"], dtype, ambiguity_eps)
    return {"proj": pf, "rec": rec, "keys": keys, "vals": vals, "ranges": ranges, "image": rf[0],
            "final_T": rf[1], "n_contrib": rf[2], "ambiguous": rf[3] if ambiguity_eps is not None else None}
