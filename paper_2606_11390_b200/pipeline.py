"""Buffer management around the C-ABI calls: one forward+backward "step" of the hot path.

This is orchestration only (allocation with torch, call order, capacity growth); all
arithmetic happens inside ``libgsplat_b200.so``.  Order of a step (SURVEY.md §3(iii),
PAPER.md:96-98):

    gs_project_fwd -> gs_bin_tiles -> gs_raster_fwd -> gs_l1_loss -> gs_raster_bwd -> gs_project_bwd
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B


class SplatStep:
    """Device-resident state for a batch of C views of one scene."""

    def __init__(self, scene, device="cuda:0", capacity_M=None, upload=True, want_keys=False):
        # want_keys: also materialise the sorted 64-bit (tile | depth) keys; no later stage reads them
        self.want_keys = bool(want_keys)
        self.device = torch.device(device)
        self.scene_name = scene.get("name", "")
        self.cams_host = scene["cameras"]
        self.cams = B.make_cameras(scene["cameras"])
        self.C = len(scene["cameras"])
        self.W, self.H = self.cams[0].width, self.cams[0].height
        self.gx, self.gy = B.grid_of(self.cams)
        self.cfg = B.default_config(sh_degree=int(scene["sh_degree"]))
        self.bg = [float(x) for x in scene["bg"]]
        self.N = int(scene["means"].shape[0])
        self.K = (self.cfg.sh_degree + 1) ** 2
        d = self.device
        f32 = torch.float32
        N, Cn = self.N, self.C
        self.param_names = ("means", "log_scales", "quats", "opacity_logits", "sh")
        self.params = {}
        shapes = {"means": (N, 3), "log_scales": (N, 3), "quats": (N, 4), "opacity_logits": (N,), "sh": (N, self.K, 3)}
        for k in self.param_names:
            self.params[k] = torch.empty(shapes[k], dtype=f32, device=d)
        if upload:
            for k in self.param_names:
                self.params[k].copy_(torch.from_numpy(np.ascontiguousarray(scene[k], dtype=np.float32)))
        self.grads = {k: torch.empty_like(v) for k, v in self.params.items()}
        # per-(view, Gaussian) records and their gradients
        self.means2d = torch.empty((Cn, N, 2), dtype=f32, device=d)
        self.depths = torch.empty((Cn, N), dtype=f32, device=d)
        self.conics = torch.empty((Cn, N, 3), dtype=f32, device=d)
        self.opacities = torch.empty((Cn, N), dtype=f32, device=d)
        self.rgbs = torch.empty((Cn, N, 3), dtype=f32, device=d)
        self.radii = torch.empty((Cn, N), dtype=torch.int32, device=d)
        self.tiles_touched = torch.empty((Cn, N), dtype=torch.int32, device=d)   # uint32 bit patterns
        self.g_means2d = torch.empty_like(self.means2d)
        self.g_conics = torch.empty_like(self.conics)
        self.g_opacities = torch.empty_like(self.opacities)
        self.g_rgbs = torch.empty_like(self.rgbs)
        # images
        self.image = torch.empty((Cn, self.H, self.W, 3), dtype=f32, device=d)
        self.final_T = torch.empty((Cn, self.H, self.W), dtype=f32, device=d)
        self.n_contrib = torch.empty((Cn, self.H, self.W), dtype=torch.int32, device=d)
        self.dL_dimage = torch.empty_like(self.image)
        self.target = None
        self.loss = torch.zeros((1,), dtype=f32, device=d)
        self.tile_ranges = torch.empty((Cn * self.gx * self.gy, 2), dtype=torch.int64, device=d)
        self.M_dev = torch.zeros((1,), dtype=torch.int64, device=d)
        self.capacity_M = 0
        self.M = None
        self._alloc_isect(capacity_M if capacity_M else max(1 << 16, 8 * Cn * N // 4))

    # -- intersection buffers ------------------------------------------------------------
    def _alloc_isect(self, capacity_M):
        self.capacity_M = int(capacity_M)
        d = self.device
        self.isect_keys = (torch.empty((self.capacity_M,), dtype=torch.int64, device=d)   # uint64 bit patterns
                           if self.want_keys else None)
        self.isect_vals = torch.empty((self.capacity_M,), dtype=torch.int32, device=d)
        nbytes = B.gs_bin_tiles_workspace_bytes(self.cfg, self.N, self.cams, self.capacity_M)
        self.workspace = torch.empty((nbytes,), dtype=torch.uint8, device=d)

    def set_target(self, target):
        t = torch.as_tensor(target, dtype=torch.float32)
        self.target = t.to(self.device).contiguous()

    # -- stages -------------------------------------------------------------------------
    def project_fwd(self):
        p = self.params
        B.gs_project_fwd(self.cfg, p["means"], p["log_scales"], p["quats"], p["opacity_logits"], p["sh"], self.cams,
                         self.means2d, self.depths, self.conics, self.opacities, self.rgbs, self.radii, self.tiles_touched)

    def bin_tiles(self, sync=True):
        """With ``sync`` the record count is read back (one host sync) and the buffers grow when
        the capacity is too small; without it the call is fully asynchronous."""
        while True:
            try:
                m = B.gs_bin_tiles(self.cfg, self.N, self.cams, self.means2d, self.depths, self.radii, self.workspace,
                                   self.capacity_M, self.isect_keys, self.isect_vals, self.tile_ranges, self.M_dev, sync)
                if sync:
                    self.M = m
                return m
            except B.GsError as e:
                if e.status != B.GS_ERR_CAPACITY:
                    raise
                self._alloc_isect(int(e.needed * 1.1) + 1024)

    def raster_fwd(self):
        B.gs_raster_fwd(self.cfg, self.cams, self.isect_vals, self.tile_ranges, self.means2d, self.conics, self.opacities,
                        self.rgbs, self.bg, self.image, self.final_T, self.n_contrib)

    def l1_loss(self):
        """The step's loss: mean L1 (reading A18, default) or, with ``loss_mode = "l1ssim"``, the fused
        0.8 L1 + 0.2 (1 - SSIM) loss of the paper's reference method (gs_l1_ssim_loss)."""
        self.loss.zero_()
        if getattr(self, "loss_mode", "l1") == "l1ssim":
            if getattr(self, "_ssim_ws", None) is None:
                nbytes = B.gs_l1_ssim_loss_workspace_bytes(self.C, self.H, self.W)
                self._ssim_ws = torch.empty((nbytes,), dtype=torch.uint8, device=self.device)
            B.gs_l1_ssim_loss(self.image, self.target, 0.2, self.dL_dimage, self.loss, self._ssim_ws)
        else:
            B.gs_l1_loss(self.image, self.target, self.dL_dimage, self.loss)

    def raster_bwd(self):
        B.gs_raster_bwd(self.cfg, self.cams, self.C * self.N, self.isect_vals, self.tile_ranges, self.means2d, self.conics,
                        self.opacities, self.rgbs, self.bg, self.final_T, self.n_contrib, self.dL_dimage, self.radii,
                        self.g_means2d, self.g_conics, self.g_opacities, self.g_rgbs)

    def project_bwd(self, accumulate=False):
        p, g = self.params, self.grads
        B.gs_project_bwd(self.cfg, p["means"], p["log_scales"], p["quats"], p["opacity_logits"], p["sh"], self.cams,
                         self.radii, self.g_means2d, self.g_conics, self.g_opacities, self.g_rgbs, g["means"],
                         g["log_scales"], g["quats"], g["opacity_logits"], g["sh"], accumulate)

    def adam(self, mode="dense", lr=0.0, beta1=0.9, beta2=0.999, eps=1e-15):
        """One fused Adam step over the five parameter arrays (gs_adam_step); ``mode`` "dense" or "sparse" (only Gaussians
        visible in >= 1 view of the batch, from the saved radii)."""
        if getattr(self, "_adam_m", None) is None:
            self._adam_m = {k: torch.zeros_like(v) for k, v in self.params.items()}
            self._adam_v = {k: torch.zeros_like(v) for k, v in self.params.items()}
            self._adam_t = 0
        self._adam_t += 1
        if mode == "sparse":
            ks = self.param_names
            B.gs_adam_step_visible([self.params[k] for k in ks], [self.grads[k] for k in ks], [self._adam_m[k] for k in ks],
                                   [self._adam_v[k] for k in ks], lr, beta1, beta2, eps, self._adam_t, self.radii)
            return
        for k in self.param_names:
            B.gs_adam_step(self.params[k], self.grads[k], self._adam_m[k], self._adam_v[k], lr, beta1, beta2, eps, self._adam_t)

    # -- whole passes -------------------------------------------------------------------
    def forward(self, sync=True):
        self.project_fwd()
        self.bin_tiles(sync)
        self.raster_fwd()

    def backward(self):
        self.raster_bwd()
        self.project_bwd()

    def step(self, sync=False):
        """One forward+backward pass with the L1 loss against ``self.target``."""
        self.forward(sync)
        self.l1_loss()
        self.backward()

    def step_from_host(self, host_params, host_target, host_loss):
        """End-to-end step: parameters and target images come from (pinned) host tensors, the loss goes back
        to ``host_loss``.  The parameters are copied on the compute stream; the target images, which only
        the loss needs, are copied on a second stream while P1, binning and R1 run, and the loss kernel waits
        for that copy.  Returns after the stream has drained (the loss value is then valid on the host)."""
        main = torch.cuda.current_stream(self.device)
        if getattr(self, "_copy_stream", None) is None:
            self._copy_stream = torch.cuda.Stream(self.device)
            self._target_ready = torch.cuda.Event()
        if self.target is None:
            self.target = torch.empty(tuple(host_target.shape), dtype=torch.float32, device=self.device)
        self._copy_stream.wait_stream(main)          # the previous step's loss kernel has read the old target
        with torch.cuda.stream(self._copy_stream):
            self.target.copy_(host_target, non_blocking=True)
            self._target_ready.record(self._copy_stream)
        for k in self.param_names:
            self.params[k].copy_(host_params[k], non_blocking=True)
        self.forward(sync=False)
        main.wait_event(self._target_ready)
        self.l1_loss()
        self.backward()
        host_loss.copy_(self.loss, non_blocking=True)
        main.synchronize()

    # launches of this library's kernels in one step (memsets excluded): P1; compact, tile y-scan, x-scan,
    # ranges, histogram scan, depth-sort histogram + passes, entry offsets, tile-sort passes (+ keys); R1, L1,
    # zero rows, R2, P5
    def launches_per_step(self):
        tile_bits = max(1, int(np.ceil(np.log2(self.C * self.gx * self.gy))))
        view_bits = int(np.ceil(np.log2(self.C))) if self.C > 1 else 0
        depth_passes = 4 + (view_bits + 7) // 8
        tile_passes = min((tile_bits + 7) // 8, (tile_bits + 8) // 9)
        compact = 2 if self.C * self.N >= (1 << 24) else 1          # visibility mask + scan over the mask for large inputs
        p5 = 6 if self.N >= (1 << 22) else 1                         # dense zero-fill as five streaming launches for large N
        loss = 2 if getattr(self, "loss_mode", "l1") == "l1ssim" else 1
        return (loss - 1) + (p5 - 1) + 1 + (4 + compact) + 1 + depth_passes + 1 + tile_passes + (1 if self.want_keys else 0) + 1 + 1 + 1 + 1 + 1
