#!/usr/bin/env python
"""bench.py -- forward+backward splatting throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload object|room|block|city|tiny]
    python bench.py --impl reference ...      # the CPU oracle timed on the host cores

A "step" is one pass of the whole hot path over one batch of synthetic views:
gs_project_fwd -> gs_bin_tiles -> gs_raster_fwd -> gs_l1_loss -> gs_raster_bwd -> gs_project_bwd.
`value` = megapixels/s (C*W*H per step / device time) with inputs resident in HBM; `e2e` = the same
with the step's inputs (parameters + target images) copied from pinned host memory and the loss read
back inside the timed region.  One JSON line is printed by rank 0.

Multi-GPU: the path is "replicas only" (north_star: no sharding, no collectives):
every rank runs the same workload on its own GPU; value = total pixels of all ranks / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fwd+bwd megapixels/s"
FP32_LANES_PER_SM = 128


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="object", choices=["tiny", "object", "room", "block", "city"])
    ap.add_argument("--n", type=int, default=None, help="override the Gaussian count (debugging only)")
    ap.add_argument("--loss", default="l1", choices=["l1", "l1ssim"],
                    help="loss of the step: mean L1 (BASELINE.json configs, default) or the fused 0.8 L1 + 0.2 (1 - SSIM) (SURVEY 8(f) NEXT-1)")
    ap.add_argument("--morton", action="store_true",
                    help="reorder the Gaussian arrays along the Morton curve of the means before timing (SURVEY 8(f) NEXT-2; "
                         "one-time preprocessing, its device time is reported as morton_sort_ms, not part of a step)")
    ap.add_argument("--adam", default="none", choices=["none", "dense", "sparse"],
                    help="append the fused Adam step (SURVEY 8(f) NEXT-3) to the step, with lr = 0 so that the scene stays the same: "
                         "dense, or sparse = only Gaussians visible in the batch")
    ap.add_argument("--sparse-grads", action="store_true",
                    help="P5 writes only the rows of Gaussians visible in the batch (gs_project_bwd accumulate = 2) instead of the dense "
                         "overwrite; goes with --adam sparse")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=20.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


# ----------------------------------------------------------------------------- peaks
def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


def load_traffic(workload, kernel):
    """DRAM bytes (read + write) per launch of `kernel` on `workload` from the committed ncu --set full
    summary (profiles/dram_traffic.csv: workload,kernel,dram_read_bytes,dram_write_bytes,source); None if absent."""
    p = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if not os.path.exists(p):
        return None
    for line in open(p):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 4 and f[0] == workload and f[1] == kernel:
            try:
                return int(float(f[2]) + float(f[3]))
            except ValueError:
                return None
    return None


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            parts = [x.strip() for x in r.split(",")]
            if len(parts) < 8:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for nme, val in zip(names, parts[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": float(max(mx)) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ----------------------------------------------------------------------------- CPU oracle leg
def oracle_sample(workload, n_override, target_seconds):
    """Time the oracle (float instantiation, single thread, as it stands) on a bounded sample of the
    workload: view by view (view 0 first, further views while the time budget allows); for each view the
    per-Gaussian stages and the binning on all N Gaussians; the per-pixel stages on every k-th tile (k
    chosen from a pilot so that one view takes at most about target_seconds), scaled by k to a full view.
    Returns MP/s for one full view (mean over the sampled views)."""
    from oracle import gs_oracle as O
    from paper_2606_11390_b200 import scenes
    O.lib()
    sc = scenes.make_scene(workload, n=n_override)
    cfg = O.make_cfg(sh_degree=sc["sh_degree"])
    f32 = np.float32
    W, H = sc["cameras"][0]["width"], sc["cameras"][0]["height"]
    gx, gy = O.grid(cfg, sc["cameras"][0])
    tiles = gx * gy
    rng = np.random.Generator(np.random.PCG64(123))
    tgt = rng.random((1, H, W, 3), dtype=f32)
    t_sum = {"project_fwd": 0.0, "bin_tiles": 0.0, "raster_fwd": 0.0, "raster_bwd": 0.0, "project_bwd": 0.0}
    full_view_s, k, n_tiles_used, cpu_s, views = [], None, 0, 0.0, 0
    for v in range(len(sc["cameras"])):
        if v > 0 and cpu_s + cpu_s / v > target_seconds:
            break
        cams = sc["cameras"][v:v + 1]
        t = {}
        t0 = time.perf_counter()
        pf = O.project_fwd(cfg, sc["means"], sc["log_scales"], sc["quats"], sc["opacity_logits"], sc["sh"], cams, f32)
        t["project_fwd"] = time.perf_counter() - t0
        t0 = time.perf_counter()
        keys, vals, ranges = O.bin_tiles(cfg, cams, pf["means2d"], pf["depths"], pf["radii"])
        t["bin_tiles"] = time.perf_counter() - t0
        lens = ranges[:, 1] - ranges[:, 0]
        if k is None:
            # pilot on a few tiles to size the sample
            pilot = np.zeros(tiles, np.uint8)
            pilot[:: max(1, tiles // 16)] = 1
            t0 = time.perf_counter()
            O.raster_fwd(cfg, cams, vals, ranges, pf["means2d"], pf["conics"], pf["opacities"], pf["rgbs"], sc["bg"], f32, tile_mask=pilot)
            tp = max(time.perf_counter() - t0, 1e-4)
            cpu_s += tp
            per_rec = tp / max(int(lens[pilot > 0].sum()), 1)
            budget = max(target_seconds - t["project_fwd"] * 2 - t["bin_tiles"], 2.0)
            est_full = per_rec * max(int(lens.sum()), 1) * 2.2          # forward + backward
            k = int(max(1, np.ceil(est_full / budget)))
        mask = np.zeros(tiles, np.uint8)
        mask[::k] = 1
        t0 = time.perf_counter()
        img, T, nc = O.raster_fwd(cfg, cams, vals, ranges, pf["means2d"], pf["conics"], pf["opacities"], pf["rgbs"], sc["bg"], f32, tile_mask=mask)
        t["raster_fwd"] = (time.perf_counter() - t0)
        dL = (np.sign(img - tgt) / img.size).astype(f32)
        t0 = time.perf_counter()
        g2 = O.raster_bwd(cfg, cams, vals, ranges, pf["means2d"], pf["conics"], pf["opacities"], pf["rgbs"], sc["bg"], T, nc, dL, f32, tile_mask=mask)
        t["raster_bwd"] = (time.perf_counter() - t0)
        t0 = time.perf_counter()
        O.project_bwd(cfg, sc["means"], sc["log_scales"], sc["quats"], sc["opacity_logits"], sc["sh"], cams, pf["radii"],
                      g2["means2d"], g2["conics"], g2["opacities"], g2["rgbs"], f32)
        t["project_bwd"] = time.perf_counter() - t0
        frac = float(mask.sum()) / tiles
        full_view_s.append(t["project_fwd"] + t["bin_tiles"] + (t["raster_fwd"] + t["raster_bwd"]) / frac + t["project_bwd"])
        for k2, val in t.items():
            t_sum[k2] += val
        cpu_s += sum(t.values())
        n_tiles_used = int(mask.sum())
        views += 1
    full_view = float(np.mean(full_view_s))
    mpix = W * H / 1e6
    return {
        "value": mpix / full_view, "unit": "MP/s", "cores": 1, "kind": "oracle",
        "sample": (f"oracle<float>, 1 thread: {views} view(s) of '{workload}' (N={sc['means'].shape[0]}), one at a time; project fwd/bwd "
                   f"and binning on all Gaussians, raster fwd+bwd on every {k}-th tile ({n_tiles_used} of {tiles}) scaled by {k}; "
                   f"measured {cpu_s:.1f} s of CPU work"),
        "stage_seconds": {k2: round(v2, 4) for k2, v2 in t_sum.items()},
        "gaussians_per_s": sc["means"].shape[0] / full_view,
        "step_mpix": len(sc["cameras"]) * mpix,
    }


def run_reference(args):
    """--impl reference: the oracle as it stands, on rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    per_step = []
    res = None
    for _ in range(args.warmup + args.steps):
        # each "step" is one bounded sample; keep the whole run within a few minutes
        res = oracle_sample(args.workload, args.n, max(2.0, min(args.cpu_seconds, 120.0 / max(args.warmup + args.steps, 1))))
        per_step.append(res["value"])
    vals = per_step[args.warmup:] or per_step
    v = float(np.mean(vals))
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": "MP/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": res["step_mpix"] / v * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": {"workload": args.workload},
        "cpu_baseline": {"value": v, "unit": "MP/s", "cores": 1, "kind": "oracle", "sample": res["sample"]},
        "e2e": {"value": v, "unit": "MP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gaussians_per_s": res["gaussians_per_s"],
    }
    print(json.dumps(line))


# ----------------------------------------------------------------------------- replicas (multi-GPU) arithmetic
def max_over_ranks(ms, world, device=None):
    """Device time of the job = the slowest rank's (all-reduce MAX over the default process group)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(world, units_per_rank_per_step, ms_per_step):
    """Replicas only: every rank processes the same units; whole-job rate = all ranks' units / max time."""
    return world * units_per_rank_per_step / (ms_per_step * 1e-3)


# ----------------------------------------------------------------------------- B200 leg
BASE_STAGES = ("project_fwd", "bin_tiles", "raster_fwd", "l1_loss", "raster_bwd", "project_bwd")


def run_b200(args):
    import torch
    import torch.distributed as dist

    from paper_2606_11390_b200 import binding as B
    from paper_2606_11390_b200 import scenes
    from paper_2606_11390_b200.pipeline import SplatStep

    B.lib()   # fails loudly when the CUDA extension is missing: there is no fallback
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)
    peaks = load_peaks()
    props = torch.cuda.get_device_properties(dev)
    sms = props.multi_processor_count

    sc = scenes.make_scene(args.workload, n=args.n)
    tgt_host = scenes.target_image(sc)
    st = SplatStep(sc, device=dev)
    st.set_target(tgt_host)
    st.loss_mode = args.loss
    morton_ms = None
    if args.morton:
        B.morton_sort({k: st.params[k] for k in st.param_names})          # warm-up (allocations, first launches)
        torch.cuda.synchronize()
        m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        m0.record()
        sorted_params, _ = B.morton_sort({k: st.params[k] for k in st.param_names})
        m1.record()
        torch.cuda.synchronize()
        morton_ms = m0.elapsed_time(m1)
        for k in st.param_names:
            st.params[k].copy_(sorted_params[k])
        del sorted_params
    C, N, W, H = st.C, st.N, st.W, st.H
    # size the intersection buffers once (one synchronising pass), then run without host syncs
    st.forward(sync=True)
    M = int(st.M)
    if st.capacity_M < M or st.capacity_M > 2 * M + (1 << 20):
        st._alloc_isect(int(M * 1.05) + 4096)
    torch.cuda.synchronize()
    flush = torch.empty((256 << 20,), dtype=torch.uint8, device=dev)     # > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    stream = torch.cuda.current_stream()

    STAGES = BASE_STAGES + (("adam",) if args.adam != "none" else ())

    def timed_step(ev):
        p5 = (lambda: st.project_bwd(accumulate=2)) if args.sparse_grads else st.project_bwd
        calls = (st.project_fwd, lambda: st.bin_tiles(sync=False), st.raster_fwd, st.l1_loss, st.raster_bwd, p5)
        if args.adam != "none":
            calls = calls + (lambda: st.adam(args.adam),)
        ev[0].record(stream)
        for k, fn in enumerate(calls):
            fn()
            ev[k + 1].record(stream)

    for _ in range(max(args.warmup, 3)):
        st.step(sync=False)
        if args.adam != "none":
            st.adam(args.adam)            # (also allocates the moments outside the timed region)
        if args.sparse_grads:
            st.project_bwd(accumulate=2)
    barrier()

    sampler = ClockSampler(local_rank)
    sampler.start()
    events = [[torch.cuda.Event(enable_timing=True) for _ in range(len(STAGES) + 1)] for _ in range(args.steps)]
    barrier()
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.fill_(k & 0xFF)                 # L2 flush between timed iterations (outside the step's events)
        timed_step(events[k])
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    step_ms = np.array([ev[0].elapsed_time(ev[-1]) for ev in events])
    stage_ms = {s: float(np.mean([ev[i].elapsed_time(ev[i + 1]) for ev in events])) for i, s in enumerate(STAGES)}
    total_ms = max_over_ranks(float(step_ms.sum()), world, dev)
    ms_per_step = total_ms / args.steps
    mpix_step = C * W * H / 1e6
    value = whole_job_rate(world, mpix_step, ms_per_step)
    gauss_per_s = whole_job_rate(world, C * N, ms_per_step)

    # ---- algorithmic work of this step (harness-side counting, outside the timed region)
    vis = st.radii > 0
    V_sum = int(vis.sum().item())
    V_any = int(vis.any(dim=0).sum().item())
    M_now = int(st.M_dev.item())
    pairs_bwd = int(st.n_contrib.to(torch.int64).sum().item())
    lens = (st.tile_ranges[:, 1] - st.tile_ranges[:, 0])
    # binning plan (mirrors gs_bin_tiles): depth sort = 4 passes over bits 0..30 plus the view bits; tile sort =
    # P_t passes of 8 or 9 bits over the tile id; the generating pass writes (key, value), the last pass values only
    tile_bits = max(1, int(np.ceil(np.log2(C * st.gx * st.gy))))
    view_bits = int(np.ceil(np.log2(C))) if C > 1 else 0
    P_d = 4 + (view_bits + 7) // 8
    P_t = min((tile_bits + 7) // 8, (tile_bits + 8) // 9)
    cells = C * (st.gx + 1) * (st.gy + 1)
    tsort_bytes = 4 * M_now if P_t == 1 else (8 + 16 * (P_t - 2) + 12) * M_now
    K3 = 3 * st.K
    par_b = 4 * (3 + 3 + 4 + 1 + K3)
    work = {
        # bytes
        "project_fwd": 12 * N + (par_b - 12) * V_any + 48 * V_sum + 8 * N * C,
        # compaction (radii; uv, depth -> key, id) + depth sort (histogram, P_d passes) + entry table + tile sort + grid scans, ranges
        "bin_tiles": 4 * N * C + 24 * V_sum + (8 + 24 * P_d) * V_sum + (32 + 16) * V_sum + tsort_bytes + 24 * cells + 16 * C * st.gx * st.gy,
        "project_bwd": 4 * N * C + 36 * V_sum + par_b * V_any + par_b * (V_any if args.sparse_grads else N),
        # L1: read image, target, write dL; L1 + SSIM: + three derivative maps written and read, image and target read twice
        "l1_loss": (12 if args.loss == "l1" else 44) * C * W * H * 3,
        # flops (per evaluated (pixel, record) pair: DESIGN.md "algorithmic flops per pair")
        # Adam: p, g, m, v read, p, m, v written, per float; sparse: radii scan + the same for visible rows only
        "adam": (28 * (par_b // 4) * N if args.adam == "dense" else 4 * N * C + 28 * (par_b // 4) * V_any),
        "raster_fwd": 22 * pairs_bwd,
        "raster_bwd": 60 * pairs_bwd,
    }
    fp32_peak = sms * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12      # TFLOP/s
    stage_roof = {}
    for s in STAGES:
        ms = stage_ms[s]
        if s in ("raster_fwd", "raster_bwd"):
            ach = work[s] / (ms * 1e-3) / 1e12
            stage_roof[s] = {"ms": round(ms, 4), "bound": "alu", "achieved": round(ach, 3), "peak": round(fp32_peak, 1),
                             "unit": "TFLOP/s", "frac": round(ach / fp32_peak, 4)}
        else:
            ach = work[s] / (ms * 1e-3) / 1e9
            stage_roof[s] = {"ms": round(ms, 4), "bound": "hbm", "achieved": round(ach, 1), "peak": peaks["hbm_gbs"],
                             "unit": "GB/s", "frac": round(ach / peaks["hbm_gbs"], 4)}
    dominant = max(STAGES, key=lambda s: stage_ms[s])
    roof = dict(stage_roof[dominant])
    roof.pop("ms")
    roof["kernel"] = {"raster_bwd": "raster_bwd_kernel", "raster_fwd": "raster_fwd_kernel", "project_fwd": "project_fwd_kernel",
                      "project_bwd": "project_bwd_kernel", "bin_tiles": "tile_sweep_kernel", "l1_loss": "l1_loss_kernel" if args.loss == "l1" else "ssim_stats_kernel",
                      "adam": "adam_dense_kernel" if args.adam == "dense" else "adam_visible_multi_kernel"}[dominant]
    roof["share_of_step"] = round(stage_ms[dominant] / (ms_per_step if world == 1 else float(step_ms.mean())), 4)
    roof["peak_source"] = ("MEASURED_PEAKS.json (%s)" % peaks["source"]) if roof["bound"] == "hbm" else \
        f"{sms} SMs x 128 FP32 lanes x 2 x {peaks['sm_max_mhz']:.0f} MHz (DESIGN.md)"
    roof["traffic"] = load_traffic(args.workload, roof["kernel"])

    # ---- end to end: inputs from pinned host memory, loss read back, every step
    e2e = None
    if not args.no_e2e:
        host_params = {k: torch.from_numpy(np.ascontiguousarray(sc[k], dtype=np.float32)).pin_memory() for k in st.param_names}
        host_tgt = torch.from_numpy(tgt_host).pin_memory()
        host_loss = torch.zeros((1,), dtype=torch.float32).pin_memory()
        h2d = sum(v.numel() * 4 for v in host_params.values()) + host_tgt.numel() * 4
        d2h = 4

        def e2e_step():
            # the public end-to-end call: H2D of parameters and targets (the target copy overlaps P1..R1 on a
            # second stream), the step, D2H of the loss, stream drained
            st.step_from_host(host_params, host_tgt, host_loss)

        for _ in range(3):
            e2e_step()
        barrier()
        n_e2e = max(3, min(args.steps, 10))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(n_e2e):
            e2e_step()
        e1.record(stream)
        barrier()
        e_ms = max_over_ranks(e0.elapsed_time(e1), world, dev)
        e2e = {"value": whole_job_rate(world, mpix_step, e_ms / n_e2e), "unit": "MP/s", "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": e_ms / n_e2e, "steps": n_e2e, "loss": float(host_loss.item())}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = oracle_sample(args.workload, args.n, args.cpu_seconds)
    line = {
        "metric": METRIC, "value": value, "unit": "MP/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": args.workload, "loss": args.loss, "morton": bool(args.morton), "adam": args.adam, "sparse_grads": bool(args.sparse_grads), "gaussians": N, "views": C, "width": W, "height": H, "sh_degree": st.cfg.sh_degree,
                   "intersections": M_now, "visible_entries": V_sum, "pairs_bwd": pairs_bwd,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "256 MiB buffer written between timed steps (L2 flush); per-step working set also exceeds the 126 MB L2"},
        "gaussians_per_s": gauss_per_s,
        "morton_sort_ms": morton_ms,
        "clocks": clocks,
        "e2e": e2e,
        "gpu_launches": (st.launches_per_step() + {"none": 0, "dense": 5, "sparse": 1}[args.adam]) * args.steps,
        "roofline": roof,
        "stages": stage_roof,
        "cpu_baseline": cpu,
        "wall_s_timed_region": round(t_wall, 3),
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
