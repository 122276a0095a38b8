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

    MASK_MIN_ENTRIES = 1 << 23

    def __init__(self, scene, device="cuda:0", capacity_M=None, upload=True, want_keys=False, use_mask=None):
        # want_keys: also materialise the sorted 64-bit (tile | depth) keys; no later stage reads them
        # use_mask: visibility travels between the stages as a bit mask [C, GS_VIS_WORDS(N)] written by P1 (no dense
        #   zero-fill of radii / tiles_touched, no pass over the C N radii in binning, R2, P5 and the visible-only Adam step)
        #   and P1 culls laterally with the scene-wide log-scale bound; False = every stage scans the dense radii
        self.want_keys = bool(want_keys)
        n_entries = len(scene["cameras"]) * int(scene["means"].shape[0])
        # None = automatic: the mask pays when the dense radii[C, N] are large (measured: city 6.74 -> 6.07 ms per step, block
        # 1.67 -> 1.63; at 4 M entries and below -- room, object -- the radii sit in the L2 and the mask gains nothing)
        self.use_mask = bool(use_mask) if use_mask is not None else n_entries >= self.MASK_MIN_ENTRIES
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
        self.vis_mask = torch.empty((Cn, B.vis_words(N)), dtype=torch.int32, device=d) if self.use_mask else None
        self.ls_bound = torch.empty((1,), dtype=f32, device=d) if self.use_mask else None
        self._ls_bound_valid = False
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
        # asynchronous overflow watch (step(sync=False)): M of the last asynchronous binning call, copied to pinned host
        # memory behind an event and checked at the start of the next step
        self._M_host = torch.zeros((1,), dtype=torch.int64).pin_memory()
        self._M_event = None
        self.overflow_count = 0
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
    def refresh_log_scale_bound(self):
        """Recompute the scene-wide log-scale bound (after the parameters were replaced; the Adam step keeps it current)."""
        if self.use_mask:
            B.gs_log_scale_bound(self.params["log_scales"], self.ls_bound)
            self._ls_bound_valid = True

    def project_fwd(self):
        p = self.params
        if self.use_mask and not self._ls_bound_valid:
            self.refresh_log_scale_bound()
        if getattr(self, "_grad_mask_swap", False):
            # project_bwd_incremental needs the mask of its last call until its next one: this P1 writes into the other buffer
            self.vis_mask, self._grad_mask = self._grad_mask, self.vis_mask
            self._grad_mask_swap = False
            self._grad_mask_valid = True
        B.gs_project_fwd(self.cfg, p["means"], p["log_scales"], p["quats"], p["opacity_logits"], p["sh"], self.cams,
                         self.means2d, self.depths, self.conics, self.opacities, self.rgbs, self.radii, self.tiles_touched,
                         vis_mask=self.vis_mask, log_scale_bound=self.ls_bound)

    def visible(self):
        """Harness-side view of the visibility as a bool tensor [C, N] (torch ops; not part of the hot path)."""
        if not self.use_mask:
            return self.radii > 0
        bits = torch.arange(32, device=self.device, dtype=torch.int32)
        m = ((self.vis_mask.unsqueeze(-1) >> bits) & 1).to(torch.bool).reshape(self.C, -1)
        return m[:, : self.N]

    def radii_dense(self):
        """Harness-side: radii with the entries of culled Gaussians set to 0 (in mask mode P1 leaves them unwritten)."""
        return torch.where(self.visible(), self.radii, torch.zeros_like(self.radii)) if self.use_mask else self.radii

    def tiles_dense(self):
        """Harness-side: tiles_touched (uint32 bit patterns in an int32 tensor) with the entries of culled Gaussians set to 0."""
        return torch.where(self.visible(), self.tiles_touched, torch.zeros_like(self.tiles_touched)) if self.use_mask else self.tiles_touched

    def check_overflow(self, wait=False):
        """Looks at the record count of the last asynchronous binning call (without blocking unless ``wait``).  When it
        exceeded the capacity, that step rendered only the background (gs_bin_tiles clears every range on overflow):
        the buffers are regrown for the following steps, ``overflow_count`` is incremented and True is returned."""
        ev = self._M_event
        if ev is None:
            return False
        if wait:
            ev.synchronize()
        elif not ev.query():
            return False
        self._M_event = None
        m = int(self._M_host.item())
        if m > self.capacity_M:
            torch.cuda.current_stream(self.device).synchronize()     # no kernel may still use the old buffers
            self._alloc_isect(int(m * 1.1) + 1024)
            self.overflow_count += 1
            return True
        return False

    def bin_tiles(self, sync=True):
        """With ``sync`` the record count is read back (one host sync) and the buffers grow when
        the capacity is too small; without it the call is fully asynchronous and the count is copied to pinned host
        memory behind an event (see ``check_overflow``)."""
        if not sync:
            self.check_overflow()
        while True:
            try:
                m = B.gs_bin_tiles(self.cfg, self.N, self.cams, self.means2d, self.depths, self.radii, self.workspace,
                                   self.capacity_M, self.isect_keys, self.isect_vals, self.tile_ranges, self.M_dev, sync,
                                   vis_mask=self.vis_mask, tile_sort=getattr(self, "tile_sort", 0))
                if sync:
                    self.M = m
                    if getattr(self, "tile_sort", 0) in (0, 1) and not getattr(self, "tile_sort_fixed", False):
                        # the two-level tile sort pays when an entry covers many tiles; with the counts of this synchronising
                        # call on the host (M, and V from the workspace header) choose for the following asynchronous calls:
                        # city without a far plane has 2.1 records per entry and is 10 ms faster with the one-level sort
                        V = int(self.workspace[8:16].view(torch.int64).item())
                        self.tile_sort = 1 if (V > 0 and m < 6 * V) else 0
                elif self._M_event is None:
                    self._M_host.copy_(self.M_dev, non_blocking=True)
                    self._M_event = torch.cuda.Event()
                    self._M_event.record(torch.cuda.current_stream(self.device))
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

    # Without the visibility mask, up to this many (view, Gaussian) entries the 2-D gradient arrays are zero-filled densely
    # (radii = NULL: four memsets, 36 bytes per entry) instead of row by row from the radii: on the small scenes a large
    # part of the entries is visible and the scattered 36-byte rows cost more than the dense stores (room, 4 M entries,
    # 39 % visible: 98 -> 27 us; object 31 -> 9 us).  P5 reads the rows of visible entries only, so it sees no difference.
    DENSE_ZERO_MAX_ENTRIES = 1 << 22

    def raster_bwd(self):
        radii = None if (not self.use_mask and self.C * self.N <= self.DENSE_ZERO_MAX_ENTRIES) else self.radii
        B.gs_raster_bwd(self.cfg, self.cams, self.C * self.N, self.isect_vals, self.tile_ranges, self.means2d, self.conics,
                        self.opacities, self.rgbs, self.bg, self.final_T, self.n_contrib, self.dL_dimage, radii,
                        self.g_means2d, self.g_conics, self.g_opacities, self.g_rgbs, vis_mask=self.vis_mask)

    def project_bwd(self, accumulate=False):
        p, g = self.params, self.grads
        B.gs_project_bwd(self.cfg, p["means"], p["log_scales"], p["quats"], p["opacity_logits"], p["sh"], self.cams,
                         self.radii, self.g_means2d, self.g_conics, self.g_opacities, self.g_rgbs, g["means"],
                         g["log_scales"], g["quats"], g["opacity_logits"], g["sh"], accumulate, vis_mask=self.vis_mask)
        if getattr(self, "_grad_mask", None) is not None:
            self._grad_mask_swap = True        # the rows written last are those of this mask (see project_bwd_incremental)

    def project_bwd_incremental(self):
        """P5 with the DENSE result (what ``project_bwd(accumulate=0)`` leaves in ``self.grads``, zeros included, bit for bit)
        without the dense zero-fill: the gradient arrays persist from step to step, so their only non-zero rows are those the
        previous call wrote.  Those rows are cleared from the previous call's visibility mask (gs_grad_zero_rows), then the
        visible rows of this step are overwritten (accumulate = 2): 2 x 236 bytes per visible Gaussian instead of 236 bytes
        for every Gaussian.  Needs the visibility mask; the first call zero-fills once.  Nothing else may write to
        ``self.grads`` between calls."""
        assert self.use_mask, "project_bwd_incremental needs the visibility mask (use_mask=True)"
        g = self.grads
        if getattr(self, "_grad_mask", None) is None:
            B.gs_grad_zero_fill(self.cfg.sh_degree, g["means"], g["log_scales"], g["quats"], g["opacity_logits"], g["sh"])
            self._grad_mask = torch.empty_like(self.vis_mask)
            self._grad_mask_valid = False
        elif self._grad_mask_valid:
            B.gs_grad_zero_rows(self.cfg.sh_degree, self.C, self._grad_mask, g["means"], g["log_scales"], g["quats"],
                                g["opacity_logits"], g["sh"])
            self._grad_mask_valid = False      # (a second call before the next P1 overwrites the same rows again)
        self.project_bwd(accumulate=2)         # (marks vis_mask as "the mask of the last call": kept until the next call)

    def adam(self, mode="dense", lr=0.0, beta1=0.9, beta2=0.999, eps=1e-15):
        """One fused Adam step over the five parameter arrays (gs_adam_step); ``mode`` "dense" (the paper's _fused_adam_,
        PAPER.md:82; needs the dense gradient, i.e. ``project_bwd(accumulate=0)``: with accumulate = 2 the rows of invisible
        Gaussians hold stale values) or "sparse" (reading A28, a SEMANTIC VARIANT: only Gaussians visible in >= 1 view of the
        batch are updated, the moments of all other rows do not decay)."""
        if getattr(self, "_adam_m", None) is None:
            self._adam_m = {k: torch.zeros_like(v) for k, v in self.params.items()}
            self._adam_v = {k: torch.zeros_like(v) for k, v in self.params.items()}
            self._adam_t = 0
        self._adam_t += 1
        if mode == "sparse":
            ks = self.param_names
            B.gs_adam_step_visible([self.params[k] for k in ks], [self.grads[k] for k in ks], [self._adam_m[k] for k in ks],
                                   [self._adam_v[k] for k in ks], lr, beta1, beta2, eps, self._adam_t,
                                   None if self.use_mask else self.radii, vis_mask=self.vis_mask, n_views=self.C,
                                   running_max=self.ls_bound, max_array=ks.index("log_scales"))
            return
        for k in self.param_names:
            B.gs_adam_step(self.params[k], self.grads[k], self._adam_m[k], self._adam_v[k], lr, beta1, beta2, eps, self._adam_t,
                           running_max=self.ls_bound if k == "log_scales" else None)

    # -- whole passes -------------------------------------------------------------------
    def forward(self, sync=True):
        self.project_fwd()
        self.bin_tiles(sync)
        self.raster_fwd()

    def backward(self):
        self.raster_bwd()
        self.project_bwd()

    # The dense zero-fill of the gradient arrays (236 N bytes at SH degree 3, the largest single item of a city step) can run
    # on a second stream underneath the rasterisation kernels, with P5 accumulating into it.  Measured on B200 (city, 60 M):
    # no gain -- 6.09 / 6.22 ms per step with the overlap (full-size grid / two persistent blocks per SM) against 6.07 ms
    # without: the 7.6 TB/s store stream saturates the HBM and the L2, and the gather latency of the rasterisation kernels
    # (R1 0.83 -> 2.8 ms while it runs) grows by what the overlap saves.  Off by default; kept for measurement.
    def fork_grad_zero_fill(self, t0=None, t1=None):
        """Start the dense zero-fill of the gradient arrays on the side stream (after everything enqueued so far);
        ``t0``/``t1``: optional timing events recorded around it on the side stream."""
        main = torch.cuda.current_stream(self.device)
        if getattr(self, "_zf_stream", None) is None:
            self._zf_stream = torch.cuda.Stream(self.device, priority=self.ZERO_FILL_STREAM_PRIORITY)
            self._zf_fork = torch.cuda.Event()
            self._zf_join = torch.cuda.Event()
        self._zf_fork.record(main)
        zs = self._zf_stream
        zs.wait_event(self._zf_fork)
        g = self.grads
        if t0 is not None:
            t0.record(zs)
        B.gs_grad_zero_fill(self.cfg.sh_degree, g["means"], g["log_scales"], g["quats"], g["opacity_logits"], g["sh"], stream=zs)
        if t1 is not None:
            t1.record(zs)
        self._zf_join.record(zs)

    def join_grad_zero_fill(self):
        torch.cuda.current_stream(self.device).wait_event(self._zf_join)

    def step(self, sync=False, overlap_zero_fill=False):
        """One forward+backward pass with the L1 loss against ``self.target``.  ``overlap_zero_fill``: zero-fill the gradients
        on a second stream while R1, the loss and R2 run (see above: no gain measured)."""
        self.project_fwd()
        self.bin_tiles(sync)
        if overlap_zero_fill:
            self.fork_grad_zero_fill()
        self.raster_fwd()
        self.l1_loss()
        self.raster_bwd()
        if overlap_zero_fill:
            self.join_grad_zero_fill()
            self.project_bwd(accumulate=1)
        else:
            self.project_bwd()

    # Every stage call is asynchronous and the record counts stay on the device, so a whole step is a fixed sequence of
    # kernel launches that can be captured once and replayed as ONE CUDA graph launch (the programmatic dependent launches
    # of launch_chained become programmatic edges of the graph).
    def capture_step_graph(self):
        """Capture one asynchronous step (P1, binning, R1, loss, R2, P5 with the dense gradient) on the current buffers into
        a CUDA graph; ``replay_step_graph`` then runs a step with one launch.  The buffers, the cameras and the record
        capacity are baked in: call again after ``set_cameras`` / a capacity change.  Overflow is reported only through
        ``graph_record_count`` (the graph never synchronises)."""
        self.step(sync=True)                 # sizes the buffers, fixes the tile-sort mode, sets every lazy kernel attribute
        torch.cuda.current_stream(self.device).synchronize()
        self._M_event = None
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            self.project_fwd()
            B.gs_bin_tiles(self.cfg, self.N, self.cams, self.means2d, self.depths, self.radii, self.workspace, self.capacity_M,
                           self.isect_keys, self.isect_vals, self.tile_ranges, self.M_dev, False, vis_mask=self.vis_mask,
                           tile_sort=getattr(self, "tile_sort", 0))
            self.raster_fwd()
            self.l1_loss()
            self.raster_bwd()
            self.project_bwd()
        self._graph = g
        self._graph_capacity = self.capacity_M
        return g

    def replay_step_graph(self):
        assert getattr(self, "_graph", None) is not None and self._graph_capacity == self.capacity_M, "capture_step_graph first"
        self._graph.replay()

    def graph_record_count(self):
        """Record count M of the last replayed step (synchronises); M > capacity_M means that step rendered only the background."""
        return int(self.M_dev.item())

    def step_from_host(self, host_params, host_target, host_loss):
        """End-to-end step, synchronous form: ``upload_async`` + ``step_uploaded`` + wait.  Parameters and target images
        come from (pinned) host tensors, the loss goes back to ``host_loss``."""
        self.upload_async(host_params, host_target)
        self.step_uploaded(host_loss)
        torch.cuda.current_stream(self.device).synchronize()

    # The end-to-end path is torch copies plus the stage calls (there is no host-buffer entry point in the C ABI).  Inputs
    # are double-buffered: upload_async(k + 1) runs on a copy stream while step k computes on the main stream.
    def upload_async(self, host_params, host_target):
        """Enqueue the H2D copies of one step's inputs (parameter arrays -- pass None to keep the resident parameters --
        and target images) into the set of device buffers that the step after the current one will use."""
        main = torch.cuda.current_stream(self.device)
        if getattr(self, "_copy_stream", None) is None:
            self._copy_stream = torch.cuda.Stream(self.device)
            self._slot = 0                       # buffer set the NEXT step_uploaded will consume
            self._pending = 0                    # uploads enqueued and not yet consumed (0..2)
            self._in_params = [None, None]
            self._in_target = [None, None]
            self._in_ready = [None, None]        # copy finished (copy stream)
            self._in_free = [None, None]         # the step that read this set has finished (main stream)
        assert self._pending < 2, "two uploads are already waiting"
        k = (self._slot + self._pending) % 2
        if self._in_target[k] is None:
            self._in_target[k] = torch.empty(tuple(host_target.shape), dtype=torch.float32, device=self.device)
            if host_params is not None:
                # set 0 is the resident parameter set itself; set 1 is a second copy
                self._in_params[k] = self.params if k == 0 else {n: torch.empty_like(v) for n, v in self.params.items()}
        cs = self._copy_stream
        if self._in_free[k] is not None:
            cs.wait_event(self._in_free[k])
        else:
            cs.wait_stream(main)
        with torch.cuda.stream(cs):
            if host_params is not None:
                for n in self.param_names:
                    self._in_params[k][n].copy_(host_params[n], non_blocking=True)
            self._in_target[k].copy_(host_target, non_blocking=True)
            ev = torch.cuda.Event()
            ev.record(cs)
        self._in_ready[k] = ev
        self._in_has_params = host_params is not None
        self._pending += 1

    def step_uploaded(self, host_loss=None):
        """Run one step on the oldest uploaded input set; the loss is copied to ``host_loss`` (pinned) asynchronously.
        Does not synchronise the host."""
        assert getattr(self, "_pending", 0) > 0, "call upload_async first"
        main = torch.cuda.current_stream(self.device)
        k = self._slot
        main.wait_event(self._in_ready[k])
        if self._in_params[k] is not None:
            self.params = self._in_params[k]
            self._ls_bound_valid = False          # new parameter values: the log-scale bound is recomputed (one reduction)
        self.target = self._in_target[k]
        self.forward(sync=False)
        self.l1_loss()
        self.backward()
        ev = torch.cuda.Event()
        ev.record(main)
        self._in_free[k] = ev
        if host_loss is not None:
            host_loss.copy_(self.loss, non_blocking=True)
        self._slot = (k + 1) % 2
        self._pending -= 1

    # launches of this library's kernels in one step (memsets excluded): P1; compact, tile y-scan, x-scan,
    # ranges, histogram scan, depth-sort histogram + passes, entry offsets, tile-sort passes (+ keys); R1, L1,
    # zero rows, R2, P5
    def launches_per_step(self, p5_launches=None):
        tile_bits = max(1, int(np.ceil(np.log2(self.C * self.gx * self.gy))))
        view_bits = int(np.ceil(np.log2(self.C))) if self.C > 1 else 0
        depth_passes = 4 + (view_bits + 7) // 8
        tile_passes = min((tile_bits + 7) // 8, (tile_bits + 8) // 9)
        # two-level tile sort (mirrors gs_bin_tiles with tile_sort = 0): group records sorted + count, scan and expansion kernels
        extra = 0
        if getattr(self, "tile_sort", 0) in (0, 2, 3) and (self.capacity_M >= (4 << 20) or getattr(self, "tile_sort", 0) in (2, 3)):
            shift = 2
            if self.C * ((self.gx + 3) // 4) * ((self.gy + 3) // 4) > 8192 or self.capacity_M >= 512 * self.C * self.gx * self.gy or getattr(self, "tile_sort", 0) == 3:
                shift = 3
            if getattr(self, "tile_sort", 0) == 2:
                shift = 2
            side = 1 << shift
            groups = self.C * ((self.gx + side - 1) // side) * ((self.gy + side - 1) // side)
            if groups <= 8192:
                gbits = max(1, int(np.ceil(np.log2(groups))))
                tile_passes = min((gbits + 7) // 8, (gbits + 8) // 9)
                extra = 3
        compact = 2 if self.use_mask else (2 if self.C * self.N >= (1 << 24) else 1)   # mask: id compaction + entry_fill_kernel;   # radii mode, large inputs: visibility mask + scan over it
        p5 = 6 if self.N >= (1 << 22) else 1                         # dense zero-fill as five streaming launches for large N
        if p5_launches is not None:
            p5 = p5_launches                                         # e.g. 2 for project_bwd_incremental (row clearing + P5)
        loss = 2 if getattr(self, "loss_mode", "l1") == "l1ssim" else 1
        zero2d = 0 if (not self.use_mask and self.C * self.N <= self.DENSE_ZERO_MAX_ENTRIES) else 1   # memsets are not counted
        return (zero2d - 1) + extra + (loss - 1) + (p5 - 1) + 1 + (4 + compact) + 1 + depth_passes + 1 + tile_passes + (1 if self.want_keys else 0) + 1 + 1 + 1 + 1 + 1
