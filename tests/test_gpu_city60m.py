"""GPU parity at the FULL city size (BASELINE.json configs[4]: 60 M Gaussians, four 4K street views), in the launch
configuration bench.py times, with the primary far plane (120 m) and without one (SURVEY.md 8(c) reading A4: far = +inf
is the reported stress variant -- tens of millions of records per view, horizon tiles with >= 1e4 entries, the load
imbalance case of PAPER.md:172-174, :215).  This is the only size where element offsets exceed 2^31 (N * 48 SH floats).

The oracle cannot run 60 M Gaussians x 4 views in the test budget, so (as in test_gpu_fullsize.py):
* P1 and P5 are per-Gaussian: the oracle runs on a ROW SUBSET (a stride over all rows, the last million rows -- beyond
  the 2^31 element offset -- and every Gaussian the CUDA path found visible) and those rows of the full-size CUDA output
  are compared; rows outside the visible set must be exactly zero in the dense gradient (checked on all 60 M rows);
* binning: properties that hold at any size on the whole output, plus sampled tile lists rebuilt from the definition;
* R1 / R2: sampled tiles (a stride plus the longest lists) with the oracle's tile mask, the oracle fed the CUDA path's
  records and lists (stage isolation).  The records are handed to the oracle in compacted form (only entries that occur
  in a list, ids renumbered): the oracle indexes records by list value, so this is a relabelling, not arithmetic.
Bars as everywhere (north_star): integer work bit-exact, image 1e-4 per channel, gradients rel. L2 1e-3.
Results are appended to gpurun_out/parity_city60m.jsonl (summarised under profiles/).
"""
import json
import os
import time

import numpy as np
import pytest

from paper_2606_11390_b200 import scenes

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

AMB_EPS = 2e-5
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def rel_l2(a, b):
    a = np.asarray(a, np.float64).ravel(); b = np.asarray(b, np.float64).ravel()
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-30))


def record(entry):
    try:
        d = os.path.join(ROOT, "gpurun_out")
        os.makedirs(d, exist_ok=True)
        with open(os.path.join(d, "parity_city60m.jsonl"), "a") as f:
            f.write(json.dumps(entry) + "\n")
    except OSError:
        pass


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_11390_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def city60():
    return scenes.make_scene("city")          # 60 M Gaussians, 14.16 GB of parameters


@pytest.mark.parametrize("far", [120.0, scenes.FAR_INF], ids=["far120", "farinf"])
def test_city_60m(B, oracle, city60, far):
    from paper_2606_11390_b200.pipeline import SplatStep
    from test_gpu_fullsize import check_project_fwd_arrays, tile_list_from_definition
    t_start = time.time()
    sc = dict(city60)
    sc["cameras"] = [dict(c, far=float(far)) for c in city60["cameras"]]
    cams = sc["cameras"]
    cfg = oracle.make_cfg(sh_degree=sc["sh_degree"])
    C, N = len(cams), sc["means"].shape[0]
    assert N == 60_000_000 and N * 48 > 2 ** 31

    # ---- the step as bench.py launches it
    st = SplatStep(sc)
    st.set_target(scenes.target_image(sc))
    st.forward(sync=True)
    M = int(st.M)
    st._alloc_isect(int(M * 1.05) + 4096)
    st.step(sync=False)
    torch.cuda.synchronize()
    assert int(st.M_dev.item()) == M and st.overflow_count == 0
    gx, gy = st.gx, st.gy
    tiles = gx * gy

    # ---- row subset for the per-Gaussian stages
    vis_t = st.visible()                                             # [C, N] on the device
    anyvis_t = vis_t.any(dim=0)
    V_sum, V_any = int(vis_t.sum().item()), int(anyvis_t.sum().item())
    stride = 4001
    rows_vis = torch.nonzero(anyvis_t).reshape(-1).cpu().numpy()
    if len(rows_vis) > 400_000:                                      # far = +inf: a third of the scene is visible
        rows_vis = rows_vis[:: len(rows_vis) // 400_000 + 1]
    rows = np.unique(np.concatenate([np.arange(0, N, stride), np.arange(N - 1_000_000, N), rows_vis])).astype(np.int64)
    rows_t = torch.from_numpy(rows).to(st.device)
    sub = {k: np.ascontiguousarray(sc[k][rows]) for k in ("means", "log_scales", "quats", "opacity_logits", "sh")}
    ref = oracle.project_fwd(cfg, sub["means"], sub["log_scales"], sub["quats"], sub["opacity_logits"], sub["sh"], cams)
    got = {k: getattr(st, k)[:, rows_t].cpu().numpy() for k in ("means2d", "depths", "conics", "opacities", "rgbs")}
    zero = torch.zeros((), dtype=torch.int32, device=st.device)
    got["radii"] = torch.where(vis_t[:, rows_t], st.radii[:, rows_t], zero).cpu().numpy()       # culled entries are unwritten in mask mode
    got["tiles_touched"] = torch.where(vis_t[:, rows_t], st.tiles_touched[:, rows_t], zero).cpu().numpy().view(np.uint32)
    p1 = check_project_fwd_arrays(got, ref, "city-60M", dict(sc, means=sub["means"], log_scales=sub["log_scales"], quats=sub["quats"]))
    del ref

    # ---- binning: properties on the whole output
    ranges = st.tile_ranges.cpu().numpy()
    lens = ranges[:, 1] - ranges[:, 0]
    nz = lens > 0
    assert lens.min() >= 0 and int(lens.sum()) == M
    assert np.all(ranges[~nz] == 0)
    starts = ranges[nz, 0]
    assert starts[0] == 0 and np.array_equal(starts[1:], ranges[nz, 1][:-1]) and ranges[nz, 1][-1] == M
    assert int(torch.where(vis_t, st.tiles_touched, zero).to(torch.int64).sum().item()) == M
    vals_t = st.isect_vals[:M].to(torch.int64)
    d_sorted = st.depths.reshape(-1)[vals_t]
    inside = torch.ones((M,), dtype=torch.bool, device=st.device)
    inside[torch.from_numpy(starts).to(st.device)] = False
    assert bool(((d_sorted[1:] >= d_sorted[:-1]) | ~inside[1:]).all())          # depth never decreases inside a list
    view_of = (vals_t // N)
    tile_view = torch.repeat_interleave(torch.arange(C * tiles, device=st.device) // tiles, torch.from_numpy(lens).to(st.device))
    assert bool((view_of == tile_view).all())                                      # every record sits in a list of its own view
    del d_sorted, inside, view_of, tile_view

    # ---- sampled tiles: a stride plus the longest lists
    sample = np.unique(np.concatenate([np.arange(0, C * tiles, 1013), np.argsort(lens)[-6:]]))
    vals = st.isect_vals[:M].cpu().numpy()
    vis_rows = [torch.nonzero(vis_t[c]).reshape(-1) for c in range(C)]              # visible Gaussians per view (device)
    per_view = []
    for c in range(C):
        r_ = vis_rows[c]
        per_view.append((r_.cpu().numpy(), st.means2d[c, r_].cpu().numpy(), st.depths[c, r_].cpu().numpy(), st.radii[c, r_].cpu().numpy()))
    n_lists = 0
    for bt in sample[:: max(1, len(sample) // 40)].tolist() + np.argsort(lens)[-2:].tolist():
        view, t = divmod(int(bt), tiles)
        idx, m2, dep, rad = per_view[view]
        # the definition restricted to the view's visible Gaussians (radius > 0); ids mapped back to entry numbers
        want_local = tile_list_from_definition(t, 0, 0, gx, gy, m2[None], dep[None], rad[None])
        want = (view * N + idx[want_local]).astype(np.int32)
        np.testing.assert_array_equal(vals[ranges[bt, 0]:ranges[bt, 1]], want)
        n_lists += 1

    # ---- R1 / R2 on the sampled tiles, oracle fed the CUDA path's records and lists (compacted)
    mask = np.zeros(C * tiles, np.uint8)
    mask[sample] = 1
    sel = np.concatenate([np.arange(ranges[bt, 0], ranges[bt, 1]) for bt in sample]) if len(sample) else np.zeros(0, np.int64)
    uniq = np.unique(vals[sel])
    vals_c = np.zeros_like(vals)
    vals_c[sel] = np.searchsorted(uniq, vals[sel]).astype(np.int32)
    uniq_t = torch.from_numpy(uniq.astype(np.int64)).to(st.device)
    rec = {"means2d": st.means2d.reshape(-1, 2)[uniq_t].cpu().numpy(), "conics": st.conics.reshape(-1, 3)[uniq_t].cpu().numpy(),
           "opacities": st.opacities.reshape(-1)[uniq_t].cpu().numpy(), "rgbs": st.rgbs.reshape(-1, 3)[uniq_t].cpu().numpy()}
    img, T, nc, amb = oracle.raster_fwd(cfg, cams, vals_c, ranges, rec["means2d"], rec["conics"], rec["opacities"], rec["rgbs"],
                                        sc["bg"], ambiguity_eps=AMB_EPS, tile_mask=mask)
    H, W = st.H, st.W
    tm = mask.reshape(C, gy, gx).astype(bool)
    pm = np.repeat(np.repeat(tm, 16, axis=1), 16, axis=2)[:, :H, :W]
    gi, gT, gn = st.image.cpu().numpy(), st.final_T.cpu().numpy(), st.n_contrib.cpu().numpy()
    clear = pm & (amb == 0)
    err = np.abs(gi - img).max(axis=-1)
    assert err[clear].max() <= 1e-4, err[clear].max()
    assert np.abs(gT - T)[clear].max() <= 1e-4
    assert np.array_equal(gn[clear], nc[clear])
    if (pm & ~clear).any():
        assert err[pm & (amb != 0)].max() <= 2e-2
    assert clear.sum() > 0.99 * pm.sum()
    rng = np.random.default_rng(5)
    dL = np.zeros((C, H, W, 3), np.float32)
    dL[pm] = (rng.standard_normal((int(pm.sum()), 3)) / (H * W)).astype(np.float32)
    st.dL_dimage.copy_(torch.from_numpy(dL))
    st.raster_bwd()
    st.project_bwd()
    torch.cuda.synchronize()
    ref2 = oracle.raster_bwd(cfg, cams, vals_c, ranges, rec["means2d"], rec["conics"], rec["opacities"], rec["rgbs"], sc["bg"],
                             gT, gn, dL, tile_mask=mask)
    g2 = {"means2d": st.g_means2d.reshape(-1, 2), "conics": st.g_conics.reshape(-1, 3), "opacities": st.g_opacities.reshape(-1),
          "rgbs": st.g_rgbs.reshape(-1, 3)}
    e2 = {k: rel_l2(g2[k][uniq_t].cpu().numpy(), ref2[k]) for k in ref2}
    for k, e in e2.items():
        assert e <= 1e-3, (k, e)
    # visible entries outside the sampled lists received nothing (dL/dimage is zero on their pixels)
    touched = torch.zeros((C * N,), dtype=torch.bool, device=st.device)
    touched[uniq_t] = True
    rest = vis_t.reshape(-1) & ~touched
    assert float(g2["opacities"][rest].abs().max().item() if bool(rest.any()) else 0.0) == 0.0
    del touched, rest

    # ---- P5 on the row subset, fed the CUDA path's 2-D gradients; all other rows of the dense gradient are zero
    g2r = {}
    for k, v in (("means2d", st.g_means2d), ("conics", st.g_conics), ("opacities", st.g_opacities), ("rgbs", st.g_rgbs)):
        a = v[:, rows_t].cpu().numpy()
        vis_r = got["radii"] > 0
        g2r[k] = np.where(vis_r[..., None] if a.ndim == 3 else vis_r, a, 0.0)        # rows of culled entries are never read
    gp = oracle.project_bwd(cfg, sub["means"], sub["log_scales"], sub["quats"], sub["opacity_logits"], sub["sh"], cams,
                            got["radii"], g2r["means2d"], g2r["conics"], g2r["opacities"], g2r["rgbs"])
    e5 = {}
    for k in gp:
        g_full = st.grads[k].reshape(N, -1)
        e5[k] = rel_l2(g_full[rows_t].cpu().numpy().reshape(gp[k].shape), gp[k])
        assert e5[k] <= 1e-3, (k, e5[k])
        nzrow = (g_full != 0).any(dim=1)
        assert not bool((nzrow & ~anyvis_t).any()), k                                  # dense overwrite: invisible rows are zero
    entry = {"test": "city_60m", "far": "inf" if far > 1e30 else far, "N": N, "C": C, "M": M, "V_sum": V_sum, "V_any": V_any,
             "rows_checked": int(len(rows)), "p1": p1, "tile_lists_exact": n_lists, "longest_list": int(lens.max()),
             "sampled_tiles": int(len(sample)), "pixels": int(pm.sum()), "image_max_err_clear": float(err[clear].max()),
             "ambiguous_pixels": int((pm & ~clear).sum()), "r2_rel_l2": e2, "p5_rel_l2": e5, "seconds": round(time.time() - t_start, 1)}
    record(entry)
    print(entry)
    del st
    torch.cuda.empty_cache()
