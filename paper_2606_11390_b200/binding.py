"""Thin ctypes binding of ``libgsplat_b200.so`` (C ABI in ``include/gsplat_b200.h``).

Argument marshalling only: every step of the hot path runs in the CUDA kernels behind the C
entry points.  PyTorch is used for device memory and streams.  Function names match the C
names.  There is NO CPU fallback: if the library is missing the import of a function raises,
and the functions refuse non-CUDA tensors.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgsplat_b200.so")

GS_OK, GS_ERR_INVALID_ARGUMENT, GS_ERR_CAPACITY, GS_ERR_CUDA, GS_ERR_UNSUPPORTED = 0, -1, -2, -3, -4
GS_TILE_SORT_AUTO, GS_TILE_SORT_ONE_LEVEL, GS_TILE_SORT_GROUPS_4, GS_TILE_SORT_GROUPS_8 = 0, 1, 2, 3
GS_SORT_STATIC_MAX_N = 1 << 20

EXPORTS = ["gs_config_default", "gs_status_string", "gs_project_fwd", "gs_bin_tiles", "gs_sort_pairs", "gs_sort_pairs_static",
           "gs_raster_fwd", "gs_raster_bwd", "gs_raster_pair_stats", "gs_project_bwd", "gs_grad_zero_fill", "gs_grad_zero_rows", "gs_log_scale_bound", "gs_l1_loss", "gs_l1_ssim_loss", "gs_bounds", "gs_morton_codes", "gs_gather_rows", "gs_adam_step", "gs_adam_step_visible"]


class gs_camera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("viewmat", C.c_float * 12),
                ("near_plane", C.c_float), ("far_plane", C.c_float)]


class gs_config(C.Structure):
    _fields_ = [("dilation", C.c_float), ("alpha_min", C.c_float), ("alpha_max", C.c_float),
                ("t_min", C.c_float), ("extent", C.c_float), ("tile", C.c_int32), ("sh_degree", C.c_int32)]


class GsError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: {status_string(status)} ({status})")


_lib = None


def lib():
    """Load the CUDA library; raises if it has not been built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_11390_b200.build` "
                               "(there is no CPU fallback)")
        _lib = C.CDLL(LIB_PATH)
        _lib.gs_status_string.restype = C.c_char_p
        _lib.gs_status_string.argtypes = [C.c_int]
        for name in EXPORTS:
            if name != "gs_status_string":
                getattr(_lib, name).restype = C.c_int
    return _lib


def status_string(status):
    return lib().gs_status_string(int(status)).decode()


def default_config(**kw):
    cfg = gs_config()
    rc = lib().gs_config_default(C.byref(cfg))
    if rc:
        raise GsError(rc, "gs_config_default")
    for k, v in kw.items():
        setattr(cfg, k, v)
    return cfg


def make_cameras(cams):
    """Sequence of camera dicts (see ``scenes.make_camera``) -> ctypes array of gs_camera."""
    arr = (gs_camera * len(cams))()
    for k, c in enumerate(cams):
        a = arr[k]
        a.width, a.height = int(c["width"]), int(c["height"])
        a.fx, a.fy, a.cx, a.cy = float(c["fx"]), float(c["fy"]), float(c["cx"]), float(c["cy"])
        vm = np.asarray(c["viewmat"], dtype=np.float32).reshape(12)
        for j in range(12):
            a.viewmat[j] = float(vm[j])
        a.near_plane, a.far_plane = float(c["near"]), float(c["far"])
    return arr


def grid_of(cams_arr):
    return (cams_arr[0].width + 15) // 16, (cams_arr[0].height + 15) // 16


def _ptr(t, dtype=None):
    import torch
    if t is None:
        return C.c_void_p(0)
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("expected a CUDA tensor (the library has no CPU path)")
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _stream(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _check(rc, where):
    if rc != GS_OK:
        raise GsError(rc, where)


def vis_words(N):
    """GS_VIS_WORDS(N): uint32 words per view of a visibility mask."""
    return (int(N) + 511) // 512 * 16


def _opt(t, dtype=None):
    return _ptr(t, dtype) if t is not None else None


def gs_project_fwd(cfg, means, log_scales, quats, opacity_logits, sh, cams, means2d, depths, conics, opacities, rgbs,
                   radii, tiles_touched, vis_mask=None, log_scale_bound=None, stream=None):
    """``vis_mask``: optional int32 tensor [C, vis_words(N)] (uint32 bit patterns), written; ``log_scale_bound``: optional
    float32 tensor of one element (see gs_log_scale_bound)."""
    import torch
    N = means.shape[0]
    rc = lib().gs_project_fwd(C.byref(cfg), C.c_int64(N), _ptr(means, torch.float32), _ptr(log_scales, torch.float32),
                              _ptr(quats, torch.float32), _ptr(opacity_logits, torch.float32), _ptr(sh, torch.float32),
                              C.c_int32(len(cams)), cams, _ptr(means2d, torch.float32), _ptr(depths, torch.float32),
                              _ptr(conics, torch.float32), _ptr(opacities, torch.float32), _ptr(rgbs, torch.float32),
                              _ptr(radii, torch.int32), _ptr(tiles_touched), _opt(vis_mask, torch.int32),
                              _opt(log_scale_bound, torch.float32), _stream(stream))
    _check(rc, "gs_project_fwd")


def gs_log_scale_bound(log_scales, bound, stream=None):
    """bound (float32 tensor of one element) = max over all log-scales."""
    import torch
    rc = lib().gs_log_scale_bound(C.c_int64(log_scales.shape[0]), _ptr(log_scales, torch.float32), _ptr(bound, torch.float32), _stream(stream))
    _check(rc, "gs_log_scale_bound")


def gs_bin_tiles_workspace_bytes(cfg, N, cams, capacity_M):
    n = C.c_size_t(0)
    rc = lib().gs_bin_tiles(C.byref(cfg), C.c_int64(N), C.c_int32(len(cams)), cams, None, None, None, None, None, C.byref(n),
                            C.c_int64(capacity_M), None, None, None, None, None, C.c_int32(0), None)
    _check(rc, "gs_bin_tiles(size query)")
    return int(n.value)


def gs_bin_tiles(cfg, N, cams, means2d, depths, radii, workspace, capacity_M, isect_keys, isect_vals, tile_ranges,
                 M_dev=None, sync=True, stream=None, vis_mask=None, tile_sort=0):
    """``isect_keys`` may be None (the 64-bit keys are then not materialised).
    Returns M (host int) when ``sync`` is true, else None (M is then only in ``M_dev``).
    Raises GsError(GS_ERR_CAPACITY) with ``.needed`` set when capacity_M is too small."""
    import torch
    wb = C.c_size_t(workspace.numel() * workspace.element_size())
    m = C.c_int64(0)
    rc = lib().gs_bin_tiles(C.byref(cfg), C.c_int64(N), C.c_int32(len(cams)), cams, _ptr(means2d, torch.float32),
                            _ptr(depths, torch.float32), _ptr(radii, torch.int32), _opt(vis_mask, torch.int32), _ptr(workspace), C.byref(wb),
                            C.c_int64(capacity_M), _ptr(isect_keys) if isect_keys is not None else None,
                            _ptr(isect_vals, torch.int32),
                            _ptr(tile_ranges, torch.int64), _ptr(M_dev, torch.int64) if M_dev is not None else None,
                            C.byref(m) if sync else None, C.c_int32(int(tile_sort)), _stream(stream))
    if rc == GS_ERR_CAPACITY:
        err = GsError(rc, "gs_bin_tiles")
        err.needed = int(m.value)
        raise err
    _check(rc, "gs_bin_tiles")
    return int(m.value) if sync else None


def gs_sort_pairs_workspace_bytes(n):
    b = C.c_size_t(0)
    rc = lib().gs_sort_pairs(C.c_int64(n), C.c_int32(64), C.c_int32(0), None, None, None, C.byref(b), None)
    _check(rc, "gs_sort_pairs(size query)")
    return int(b.value)


def gs_sort_pairs(n, end_bit, skip_bit31, keys, vals, workspace, stream=None):
    import torch
    wb = C.c_size_t(workspace.numel() * workspace.element_size())
    rc = lib().gs_sort_pairs(C.c_int64(n), C.c_int32(end_bit), C.c_int32(1 if skip_bit31 else 0), _ptr(keys),
                             _ptr(vals, torch.int32), _ptr(workspace), C.byref(wb), _stream(stream))
    _check(rc, "gs_sort_pairs")


def gs_sort_pairs_static(n, end_bit, skip_bit31, keys, vals, stream=None):
    """gs_sort_pairs without a workspace: the scratch is a static device array inside the library (n <= GS_SORT_STATIC_MAX_N);
    nothing is allocated.  Calls that overlap on the GPU race on that array."""
    import torch
    rc = lib().gs_sort_pairs_static(C.c_int64(n), C.c_int32(end_bit), C.c_int32(1 if skip_bit31 else 0), _ptr(keys),
                                    _ptr(vals, torch.int32), _stream(stream))
    _check(rc, f"gs_sort_pairs_static(n = {n}, limit GS_SORT_STATIC_MAX_N = {GS_SORT_STATIC_MAX_N})")


def _bg(bg):
    return (C.c_float * 3)(float(bg[0]), float(bg[1]), float(bg[2]))


def gs_raster_fwd(cfg, cams, isect_vals, tile_ranges, means2d, conics, opacities, rgbs, bg, image, final_T, n_contrib,
                  stream=None):
    import torch
    rc = lib().gs_raster_fwd(C.byref(cfg), C.c_int32(len(cams)), cams, _ptr(isect_vals, torch.int32),
                             _ptr(tile_ranges, torch.int64), _ptr(means2d, torch.float32), _ptr(conics, torch.float32),
                             _ptr(opacities, torch.float32), _ptr(rgbs, torch.float32), _bg(bg),
                             _ptr(image, torch.float32), _ptr(final_T, torch.float32), _ptr(n_contrib, torch.int32),
                             _stream(stream))
    _check(rc, "gs_raster_fwd")


def gs_raster_bwd(cfg, cams, N_total, isect_vals, tile_ranges, means2d, conics, opacities, rgbs, bg, final_T, n_contrib,
                  dL_dimage, radii, dL_dmeans2d, dL_dconics, dL_dopacities, dL_drgbs, stream=None, vis_mask=None):
    import torch
    rc = lib().gs_raster_bwd(C.byref(cfg), C.c_int32(len(cams)), cams, C.c_int64(N_total), _ptr(isect_vals, torch.int32),
                             _ptr(tile_ranges, torch.int64), _ptr(means2d, torch.float32), _ptr(conics, torch.float32),
                             _ptr(opacities, torch.float32), _ptr(rgbs, torch.float32), _bg(bg),
                             _ptr(final_T, torch.float32), _ptr(n_contrib, torch.int32), _ptr(dL_dimage, torch.float32),
                             _opt(radii, torch.int32), _opt(vis_mask, torch.int32), _ptr(dL_dmeans2d, torch.float32),
                             _ptr(dL_dconics, torch.float32), _ptr(dL_dopacities, torch.float32),
                             _ptr(dL_drgbs, torch.float32), _stream(stream))
    _check(rc, "gs_raster_bwd")


def gs_raster_pair_stats(cfg, cams, isect_vals, tile_ranges, means2d, conics, opacities, stats, stream=None):
    """Measurement aid: stats (int64[4], device) = composited pairs, pairs the forward / the backward definition evaluates
    without compositing, 256 x records."""
    import torch
    rc = lib().gs_raster_pair_stats(C.byref(cfg), C.c_int32(len(cams)), cams, _ptr(isect_vals, torch.int32),
                                    _ptr(tile_ranges, torch.int64), _ptr(means2d, torch.float32), _ptr(conics, torch.float32),
                                    _ptr(opacities, torch.float32), _ptr(stats, torch.int64), _stream(stream))
    _check(rc, "gs_raster_pair_stats")


def gs_project_bwd(cfg, means, log_scales, quats, opacity_logits, sh, cams, radii, dL_dmeans2d, dL_dconics,
                   dL_dopacities, dL_drgbs, dL_dmeans, dL_dlog_scales, dL_dquats, dL_dopacity_logits, dL_dsh,
                   accumulate=False, stream=None, vis_mask=None):
    import torch
    N = means.shape[0]
    rc = lib().gs_project_bwd(C.byref(cfg), C.c_int64(N), _ptr(means, torch.float32), _ptr(log_scales, torch.float32),
                              _ptr(quats, torch.float32), _ptr(opacity_logits, torch.float32), _ptr(sh, torch.float32),
                              C.c_int32(len(cams)), cams, _opt(radii, torch.int32), _opt(vis_mask, torch.int32), _ptr(dL_dmeans2d, torch.float32),
                              _ptr(dL_dconics, torch.float32), _ptr(dL_dopacities, torch.float32),
                              _ptr(dL_drgbs, torch.float32), _ptr(dL_dmeans, torch.float32),
                              _ptr(dL_dlog_scales, torch.float32), _ptr(dL_dquats, torch.float32),
                              _ptr(dL_dopacity_logits, torch.float32), _ptr(dL_dsh, torch.float32),
                              C.c_int32(int(accumulate)), _stream(stream))
    _check(rc, "gs_project_bwd")


def gs_grad_zero_fill(sh_degree, dL_dmeans, dL_dlog_scales, dL_dquats, dL_dopacity_logits, dL_dsh, stream=None):
    import torch
    N = dL_dmeans.shape[0]
    rc = lib().gs_grad_zero_fill(C.c_int64(N), C.c_int32(sh_degree), _ptr(dL_dmeans, torch.float32), _ptr(dL_dlog_scales, torch.float32),
                                 _ptr(dL_dquats, torch.float32), _ptr(dL_dopacity_logits, torch.float32), _ptr(dL_dsh, torch.float32),
                                 _stream(stream))
    _check(rc, "gs_grad_zero_fill")


def gs_grad_zero_rows(sh_degree, n_views, vis_mask, dL_dmeans, dL_dlog_scales, dL_dquats, dL_dopacity_logits, dL_dsh, stream=None):
    """Zero the gradient rows of the Gaussians that ``vis_mask`` ([n_views, vis_words(N)]) marks in any view."""
    import torch
    N = dL_dmeans.shape[0]
    assert vis_mask.numel() == n_views * vis_words(N)
    rc = lib().gs_grad_zero_rows(C.c_int64(N), C.c_int32(sh_degree), C.c_int32(n_views), _ptr(vis_mask), _ptr(dL_dmeans, torch.float32),
                                 _ptr(dL_dlog_scales, torch.float32), _ptr(dL_dquats, torch.float32),
                                 _ptr(dL_dopacity_logits, torch.float32), _ptr(dL_dsh, torch.float32), _stream(stream))
    _check(rc, "gs_grad_zero_rows")


def gs_l1_loss(image, target, dL_dimage, loss_sum, stream=None):
    import torch
    rc = lib().gs_l1_loss(C.c_int64(image.numel()), _ptr(image, torch.float32), _ptr(target, torch.float32),
                          _ptr(dL_dimage, torch.float32), _ptr(loss_sum, torch.float32), _stream(stream))
    _check(rc, "gs_l1_loss")


def gs_l1_ssim_loss_workspace_bytes(C_views, height, width):
    nbytes = C.c_size_t(0)
    rc = lib().gs_l1_ssim_loss(C.c_int32(C_views), C.c_int32(height), C.c_int32(width), None, None, C.c_float(0.2), None, None,
                               None, C.byref(nbytes), None)
    _check(rc, "gs_l1_ssim_loss")
    return int(nbytes.value)


def gs_l1_ssim_loss(image, target, lam, dL_dimage, loss_sum, workspace, stream=None):
    """image, target, dL_dimage: [C, H, W, 3] float32 CUDA tensors; loss_sum: 1 float (caller-zeroed, added to)."""
    import torch
    Cv, H, W, ch = image.shape
    assert ch == 3 and tuple(target.shape) == tuple(image.shape) == tuple(dL_dimage.shape)
    nbytes = C.c_size_t(workspace.numel() * workspace.element_size())
    rc = lib().gs_l1_ssim_loss(C.c_int32(Cv), C.c_int32(H), C.c_int32(W), _ptr(image, torch.float32), _ptr(target, torch.float32),
                               C.c_float(lam), _ptr(dL_dimage, torch.float32), _ptr(loss_sum, torch.float32),
                               _ptr(workspace, torch.uint8), C.byref(nbytes), _stream(stream))
    _check(rc, "gs_l1_ssim_loss")


def gs_bounds(means, lo_hi, stream=None):
    import torch
    rc = lib().gs_bounds(C.c_int64(means.shape[0]), _ptr(means, torch.float32), _ptr(lo_hi, torch.float32), _stream(stream))
    _check(rc, "gs_bounds")


def gs_morton_codes(means, lo_hi, codes, index, stream=None):
    """codes: int64 tensor holding the uint64 bit patterns; index: int32."""
    import torch
    rc = lib().gs_morton_codes(C.c_int64(means.shape[0]), _ptr(means, torch.float32), _ptr(lo_hi, torch.float32),
                               _ptr(codes, torch.int64), _ptr(index, torch.int32), _stream(stream))
    _check(rc, "gs_morton_codes")


def gs_gather_rows(src, perm, dst, stream=None):
    import torch
    N = src.shape[0]
    row = src.numel() // max(N, 1)
    rc = lib().gs_gather_rows(C.c_int64(N), C.c_int32(row), _ptr(src, torch.float32), _ptr(perm, torch.int32),
                              _ptr(dst, torch.float32), _stream(stream))
    _check(rc, "gs_gather_rows")


def morton_sort(params, stream=None):
    """Reorder the parameter tensors (dict of [N, ...] float32 CUDA tensors with key "means") along the Morton curve of the
    means.  Returns (sorted dict, perm int32[N]).  Orchestration only: bounds, codes, radix sort and gathers are kernels."""
    import torch
    means = params["means"]
    N = means.shape[0]
    dev = means.device
    lo_hi = torch.empty((6,), dtype=torch.float32, device=dev)
    codes = torch.empty((N,), dtype=torch.int64, device=dev)
    perm = torch.empty((N,), dtype=torch.int32, device=dev)
    gs_bounds(means, lo_hi, stream)
    gs_morton_codes(means, lo_hi, codes, perm, stream)
    ws = torch.empty((gs_sort_pairs_workspace_bytes(N),), dtype=torch.uint8, device=dev)
    gs_sort_pairs(N, 63, 0, codes, perm, ws, stream)
    out = {}
    for k, t in params.items():
        d = torch.empty_like(t)
        gs_gather_rows(t, perm, d, stream)
        out[k] = d
    return out, perm


def gs_adam_step(param, grad, m, v, lr, beta1, beta2, eps, step, radii=None, stream=None, running_max=None):
    """In-place Adam step on one [N, ...] float32 array; with ``radii`` ([C, N] int32) only rows visible in >= 1 view."""
    import torch
    N = param.shape[0]
    row = param.numel() // max(N, 1)
    Cv = int(radii.shape[0]) if radii is not None else 0
    rc = lib().gs_adam_step(C.c_int64(N), C.c_int32(row), _ptr(param, torch.float32), _ptr(grad, torch.float32),
                            _ptr(m, torch.float32), _ptr(v, torch.float32), C.c_float(lr), C.c_float(beta1), C.c_float(beta2),
                            C.c_float(eps), C.c_int32(step), _ptr(radii, torch.int32) if radii is not None else None,
                            C.c_int32(Cv), _opt(running_max, torch.float32), _stream(stream))
    _check(rc, "gs_adam_step")


def gs_adam_step_visible(params, grads, ms, vs, lr, beta1, beta2, eps, step, radii, stream=None, vis_mask=None, n_views=None,
                         running_max=None, max_array=0):
    """Visible-only Adam step over several [N, ...] float32 arrays (lists of tensors) in one launch; the visible rows come
    from ``vis_mask`` ([C, vis_words(N)]) when given, else from ``radii`` ([C, N])."""
    import torch
    n = len(params)
    N = params[0].shape[0]
    rows = (C.c_int32 * n)(*[t.numel() // max(N, 1) for t in params])
    def ptrs(ts):
        return (C.c_void_p * n)(*[_ptr(t, torch.float32).value for t in ts])
    rc = lib().gs_adam_step_visible(C.c_int64(N), C.c_int32(n), rows, ptrs(params), ptrs(grads), ptrs(ms), ptrs(vs), C.c_float(lr),
                                    C.c_float(beta1), C.c_float(beta2), C.c_float(eps), C.c_int32(step), _opt(radii, torch.int32),
                                    _opt(vis_mask, torch.int32), C.c_int32(int(n_views if n_views is not None else (vis_mask if radii is None else radii).shape[0])),
                                    _opt(running_max, torch.float32), C.c_int32(int(max_array)), _stream(stream))
    _check(rc, "gs_adam_step_visible")
