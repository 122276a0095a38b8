"""GPU tests of the visibility-mask path (include/gsplat_b200.h, GS_VIS_WORDS): gs_project_fwd reports visibility as a bit
mask and culls laterally with the scene-wide log-scale bound; gs_bin_tiles, gs_raster_bwd, gs_project_bwd and
gs_adam_step_visible read the mask instead of scanning the dense radii[C, N].  The mask changes no result: every check here
is against the radii path (itself compared with the oracle in test_gpu_parity.py) or against the oracle directly.
"""
import numpy as np
import pytest

from paper_2606_11390_b200 import scenes

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from test_gpu_parity import SCENES, dev, oracle_stage1, rel_l2  # noqa: E402


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_11390_b200 import binding
    binding.lib()
    return binding


def pack_mask(vis, words):
    """bool [C, N] -> uint32 words [C, words] (bit i & 31 of word i >> 5), as an int32 numpy array."""
    C, N = vis.shape
    padded = np.zeros((C, words * 32), dtype=np.uint8)
    padded[:, :N] = vis
    return np.packbits(padded.reshape(C, words, 32), axis=-1, bitorder="little").view(np.uint32).reshape(C, words).view(np.int32)


def street_scene(n=300_007):
    """A block-like scene: street-level camera with a 120 m far plane, a few per cent of the Gaussians visible."""
    sc = scenes.make_scene("block", n=n)
    cam = sc["cameras"][0]
    eye = np.asarray(cam["viewmat"])[:, :3].T @ -np.asarray(cam["viewmat"])[:, 3]
    sc["cameras"] = [scenes.make_camera(640, 360, 500.0, 500.0, eye, eye + np.array(d), (0, 0, 1), far=120.0)
                     for d in ((1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (-1.0, 0.2, 0.0))]
    return sc


MASK_SCENES = SCENES[:3] + [("street", street_scene())]


def project(B, sc, mask, bound, poison=True):
    cams = B.make_cameras(sc["cameras"])
    cfg = B.default_config(sh_degree=sc["sh_degree"])
    C, N = len(sc["cameras"]), sc["means"].shape[0]
    f32 = torch.float32
    out = {"means2d": torch.zeros((C, N, 2), dtype=f32, device="cuda"), "depths": torch.zeros((C, N), dtype=f32, device="cuda"),
           "conics": torch.zeros((C, N, 3), dtype=f32, device="cuda"), "opacities": torch.zeros((C, N), dtype=f32, device="cuda"),
           "rgbs": torch.zeros((C, N, 3), dtype=f32, device="cuda"),
           "radii": torch.full((C, N), 7777 if poison else 0, dtype=torch.int32, device="cuda"),
           "tiles_touched": torch.full((C, N), 99 if poison else 0, dtype=torch.int32, device="cuda")}
    vm = torch.full((C, B.vis_words(N)), -1, dtype=torch.int32, device="cuda") if mask else None     # all ones: must be overwritten
    lb = None
    if bound:
        lb = torch.zeros((1,), dtype=f32, device="cuda")
        B.gs_log_scale_bound(dev(sc["log_scales"]), lb)
    B.gs_project_fwd(cfg, dev(sc["means"]), dev(sc["log_scales"]), dev(sc["quats"]), dev(sc["opacity_logits"]), dev(sc["sh"]),
                     cams, out["means2d"], out["depths"], out["conics"], out["opacities"], out["rgbs"], out["radii"],
                     out["tiles_touched"], vis_mask=vm, log_scale_bound=lb)
    torch.cuda.synchronize()
    return out, vm, lb


@pytest.mark.parametrize("name,sc", MASK_SCENES, ids=[s[0] for s in MASK_SCENES])
def test_project_fwd_mask_and_bound_change_nothing(B, name, sc):
    """Mask bits == (radii > 0) of the dense call; the records of visible entries are bit-identical; entries of culled
    Gaussians are left unwritten (the poison survives); padding bits are zero; the log-scale bound drops nothing visible."""
    ref, _, _ = project(B, sc, mask=False, bound=False, poison=False)
    vis = (ref["radii"] > 0).cpu().numpy()
    C, N = vis.shape
    for bound in (False, True):
        got, vm, lb = project(B, sc, mask=True, bound=bound)
        want = pack_mask(vis, B.vis_words(N))
        np.testing.assert_array_equal(vm.cpu().numpy(), want)
        v = torch.from_numpy(vis).cuda()
        for k in ref:
            assert torch.equal(got[k][v], ref[k][v]), (k, bound)
        assert bool((got["radii"][~v] == 7777).all()) and bool((got["tiles_touched"][~v] == 99).all())
        if bound:
            assert abs(float(lb.item()) - float(sc["log_scales"].max())) == 0.0
    # bound without mask: the dense outputs are unchanged as well
    got, _, _ = project(B, sc, mask=False, bound=True, poison=True)
    assert torch.equal(got["radii"], ref["radii"]) and torch.equal(got["tiles_touched"], ref["tiles_touched"])
    print(f"[{name}] visible {int(vis.sum())} of {vis.size}")


def test_log_scale_bound_values(B):
    rng = np.random.default_rng(5)
    for n in (1, 3, 1000, 100_003):
        for shift in (-9.0, 0.0, 4.0):
            ls = (rng.standard_normal((n, 3)) + shift).astype(np.float32)
            out = torch.full((1,), 123.0, dtype=torch.float32, device="cuda")
            B.gs_log_scale_bound(dev(ls), out)
            assert float(out.item()) == float(ls.max())
    # an unaligned view takes the scalar path
    ls = (rng.standard_normal((1001, 3)) - 2.0).astype(np.float32)
    t = dev(np.concatenate([np.zeros((1, 3), np.float32), ls]))[1:]
    out = torch.zeros((1,), dtype=torch.float32, device="cuda")
    B.gs_log_scale_bound(t, out)
    assert float(out.item()) == float(ls.max())


@pytest.mark.parametrize("name,sc", MASK_SCENES[1:], ids=[s[0] for s in MASK_SCENES[1:]])
def test_bin_tiles_from_mask_bit_exact(B, oracle, name, sc):
    """Stage isolation as in test_bin_tiles_bit_exact, visibility handed over as a mask built from the ORACLE's radii; the
    radii of culled entries are poisoned to prove they are not read."""
    cfg, pf, rec = oracle_stage1(oracle, sc)
    keys, vals, ranges = oracle.bin_tiles(cfg, sc["cameras"], rec["means2d"], rec["depths"], pf["radii"])
    cams = B.make_cameras(sc["cameras"])
    bcfg = B.default_config(sh_degree=sc["sh_degree"])
    C, N = pf["radii"].shape
    gx, gy = B.grid_of(cams)
    vis = pf["radii"] > 0
    radii = np.where(vis, pf["radii"], 12345).astype(np.int32)
    vm = dev(pack_mask(vis, B.vis_words(N)))
    for cap, sync, mode in ((len(keys) + 1000, True, 0), (len(keys), False, 2), (len(keys) + 7, False, 3)):      # (tile_sort modes)
        gk = torch.zeros((cap,), dtype=torch.int64, device="cuda")
        gv = torch.zeros((cap,), dtype=torch.int32, device="cuda")
        gr = torch.full((C * gx * gy, 2), -1, dtype=torch.int64, device="cuda")
        ws = torch.empty((B.gs_bin_tiles_workspace_bytes(bcfg, N, cams, cap),), dtype=torch.uint8, device="cuda")
        M_dev = torch.full((1,), -1, dtype=torch.int64, device="cuda")
        B.gs_bin_tiles(bcfg, N, cams, dev(rec["means2d"]), dev(rec["depths"]), dev(radii), ws, cap, gk, gv, gr, M_dev, sync, vis_mask=vm,
                       tile_sort=mode)
        torch.cuda.synchronize()
        M = int(M_dev.item())
        assert M == len(keys)
        np.testing.assert_array_equal(gk.cpu().numpy().view(np.uint64)[:M], keys)
        np.testing.assert_array_equal(gv.cpu().numpy()[:M], vals)
        np.testing.assert_array_equal(gr.cpu().numpy(), ranges)
    # capacity too small: the needed size is still exact
    with pytest.raises(B.GsError) as ei:
        cap = len(keys) // 3
        ws = torch.empty((B.gs_bin_tiles_workspace_bytes(bcfg, N, cams, cap),), dtype=torch.uint8, device="cuda")
        B.gs_bin_tiles(bcfg, N, cams, dev(rec["means2d"]), dev(rec["depths"]), dev(radii), ws, cap, None,
                       torch.zeros((cap,), dtype=torch.int32, device="cuda"), gr, M_dev, True, vis_mask=vm)
    assert ei.value.status == B.GS_ERR_CAPACITY and ei.value.needed == len(keys)


@pytest.mark.parametrize("name,sc", MASK_SCENES, ids=[s[0] for s in MASK_SCENES])
def test_whole_step_mask_mode_equals_radii_mode(B, name, sc):
    """SplatStep with the mask (the default) against SplatStep scanning the dense radii: same lists, same image bit for bit,
    gradients equal up to the order of the float atomics; accumulate = 2 and the visible-only Adam step touch the same rows."""
    from paper_2606_11390_b200.pipeline import SplatStep
    tgt = scenes.target_image(sc)
    steps = []
    for use_mask in (False, True):
        st = SplatStep(sc, use_mask=use_mask)
        if use_mask:
            st.radii.fill_(31337); st.tiles_touched.fill_(-5)        # stale contents of culled entries must not matter
        st.set_target(tgt)
        st.step(sync=True)
        torch.cuda.synchronize()
        steps.append(st)
    a, b = steps
    assert a.M == b.M and a.M > 0
    assert torch.equal(a.visible(), b.visible())
    assert torch.equal(a.radii, b.radii_dense())
    assert torch.equal(a.isect_vals[: a.M], b.isect_vals[: a.M]) and torch.equal(a.tile_ranges, b.tile_ranges)
    assert torch.equal(a.image, b.image) and torch.equal(a.final_T, b.final_T) and torch.equal(a.n_contrib, b.n_contrib)
    assert abs(float(a.loss.item()) - float(b.loss.item())) <= 1e-5 * float(a.loss.item())      # (float atomics: order varies)
    vis_any = a.visible().any(dim=0)
    for k in a.grads:
        ga, gb = a.grads[k], b.grads[k]
        assert bool((gb[~vis_any] == 0).all()), k
        assert rel_l2(gb.cpu().numpy(), ga.cpu().numpy()) <= 1e-5, k
    # visible rows only (accumulate = 2) and the visible-only optimizer step
    for st in steps:
        for v in st.grads.values():
            v.fill_(0.25)
        st.project_bwd(accumulate=2)
        st.adam("sparse", lr=1e-2)
    torch.cuda.synchronize()
    for k in a.grads:
        assert bool((b.grads[k][~vis_any] == 0.25).all()), k
        assert rel_l2(b.grads[k].cpu().numpy(), a.grads[k].cpu().numpy()) <= 1e-5, k
        assert torch.equal(b.params[k][~vis_any], torch.from_numpy(np.ascontiguousarray(sc[k], dtype=np.float32)).cuda()[~vis_any]), k
        assert rel_l2(b.params[k].cpu().numpy(), a.params[k].cpu().numpy()) <= 1e-6, k
        assert not torch.equal(b.params[k][vis_any], torch.from_numpy(np.ascontiguousarray(sc[k], dtype=np.float32)).cuda()[vis_any]), k
    # the optimizer kept the log-scale bound an upper bound
    assert float(b.ls_bound.item()) >= float(b.params["log_scales"].max().item())
    print(f"[{name}] M {a.M}, visible Gaussians {int(vis_any.sum())} of {a.N}")


def test_adam_running_max(B):
    """running_max = max(running_max, updated values): it rises with the parameters and never falls."""
    rng = np.random.default_rng(11)
    n = 50_001
    p = (rng.standard_normal((n, 3)) - 3.0).astype(np.float32)
    for sign in (-1.0, 1.0):                       # gradient -1: every value rises by lr in the first step; +1: falls
        dp, dg = dev(p), dev(np.full((n, 3), sign, np.float32))
        dm, dv = torch.zeros_like(dp), torch.zeros_like(dp)
        bound = torch.full((1,), float(p.max()), dtype=torch.float32, device="cuda")
        B.gs_adam_step(dp, dg, dm, dv, 0.5, 0.9, 0.999, 1e-8, 1, running_max=bound)
        torch.cuda.synchronize()
        new_max = float(dp.max().item())
        assert (new_max > float(p.max())) == (sign < 0)
        assert float(bound.item()) == max(float(p.max()), new_max)


def test_uploaded_parameters_refresh_the_scale_bound(B):
    """The lateral cull of P1 is only valid with a bound >= every log-scale.  A second parameter set is uploaded in which some
    Gaussians far outside the image grow so large that they reach it: they are visible only if the bound was recomputed for
    the new parameters (SplatStep does that in step_uploaded); with the stale bound P1 drops them (checked as well, so that
    this test is known to see the failure)."""
    from paper_2606_11390_b200.pipeline import SplatStep
    name, sc = MASK_SCENES[3]
    sc2 = dict(sc)
    ls = sc["log_scales"].copy()
    cam = sc["cameras"][0]
    vm = np.asarray(cam["viewmat"], np.float64).reshape(3, 4)
    t = sc["means"].astype(np.float64) @ vm[:, :3].T + vm[:, 3]
    lateral = (t[:, 2] > 20) & (t[:, 2] < 100) & (np.abs(t[:, 0]) > 1.5 * t[:, 2]) & (np.abs(t[:, 0]) < 2.5 * t[:, 2])
    grown = np.nonzero(lateral)[0][:200]
    assert len(grown) >= 50
    ls[grown] = np.log(0.6 * np.abs(t[grown, 0]))[:, None].astype(np.float32)        # 3 sigma reaches the optical axis
    sc2["log_scales"] = ls
    tgt = scenes.target_image(sc)
    ref = SplatStep(sc2, use_mask=False)
    ref.set_target(tgt)
    ref.step(sync=True)
    torch.cuda.synchronize()
    vis_ref = ref.visible()
    assert bool(vis_ref[0, torch.from_numpy(grown).cuda()].any())                      # the grown Gaussians do reach view 0

    st = SplatStep(sc, use_mask=True, capacity_M=ref.capacity_M)
    st.set_target(tgt)
    st.step(sync=True)                                                                 # bound of the FIRST parameter set is now cached
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory()
    host = {k: pin(sc2[k]) for k in st.param_names}
    host_loss = torch.zeros((1,), dtype=torch.float32).pin_memory()
    st.step_from_host(host, pin(tgt), host_loss)
    torch.cuda.synchronize()
    assert float(st.ls_bound.item()) == float(ls.max())
    assert torch.equal(st.visible(), vis_ref)
    assert torch.equal(st.image, ref.image)
    # the failure this guards against: the same step with the stale bound of the first parameter set
    B.gs_log_scale_bound(dev(sc["log_scales"]), st.ls_bound)
    st.project_fwd()
    torch.cuda.synchronize()
    assert not torch.equal(st.visible(), vis_ref)


def test_incremental_gradient_clearing_equals_the_dense_overwrite(B):
    """project_bwd_incremental (gs_grad_zero_rows from the previous step's mask + gs_project_bwd accumulate = 2) must leave
    exactly the arrays of gs_project_bwd(accumulate = 0) -- zeros of the invisible rows included, bit for bit (P5 has no
    atomics; both run on the same 2-D gradients) -- over steps whose cameras, and so whose visible sets, change; also after a
    repeated call without a new P1 and after a dense call in between."""
    from paper_2606_11390_b200.pipeline import SplatStep
    sc = street_scene()
    cam = sc["cameras"][0]
    eye = np.asarray(cam["viewmat"])[:, :3].T @ -np.asarray(cam["viewmat"])[:, 3]
    dirs = [((1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (-1.0, 0.2, 0.0)), ((0.0, -1.0, 0.0), (1.0, 1.0, 0.0), (-1.0, -1.0, 0.0)),
            ((0.3, 1.0, 0.1), (-1.0, 0.0, 0.0), (1.0, -0.4, 0.0)), ((1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (-1.0, 0.2, 0.0))]
    st = SplatStep(sc, use_mask=True)
    st.set_target(scenes.target_image(sc))
    ref = {k: torch.empty_like(v) for k, v in st.grads.items()}
    for v in st.grads.values():
        v.fill_(7.5)                                         # the first call must not rely on the arrays' contents
    seen = None
    for step, d3 in enumerate(dirs):
        st.cams = B.make_cameras([scenes.make_camera(640, 360, 500.0, 500.0, eye, eye + np.array(d), (0, 0, 1), far=120.0) for d in d3])
        st.project_fwd(); st.bin_tiles(sync=True); st.raster_fwd(); st.l1_loss(); st.raster_bwd()
        p = st.params
        for v in ref.values():
            v.fill_(float("nan"))
        B.gs_project_bwd(st.cfg, p["means"], p["log_scales"], p["quats"], p["opacity_logits"], p["sh"], st.cams, st.radii,
                         st.g_means2d, st.g_conics, st.g_opacities, st.g_rgbs, ref["means"], ref["log_scales"], ref["quats"],
                         ref["opacity_logits"], ref["sh"], 0, vis_mask=st.vis_mask)
        if step == 2:
            st.project_bwd()                                 # a dense call in between keeps the bookkeeping right
        else:
            st.project_bwd_incremental()
            if step == 1:
                st.project_bwd_incremental()                 # again, without a new P1
        torch.cuda.synchronize()
        vis_any = st.visible().any(dim=0)
        n_vis = int(vis_any.sum())
        assert 0 < n_vis < st.N // 4
        if seen is not None:
            assert int((seen & ~vis_any).sum()) > 1000       # rows written before and invisible now: they must be zero again
        seen = vis_any if seen is None else (seen | vis_any)
        for k in ref:
            assert not bool(torch.isnan(ref[k]).any()), k
            assert torch.equal(st.grads[k], ref[k]), (step, k)
            assert bool((st.grads[k][~vis_any] == 0).all()), (step, k)
        print(f"[step {step}] visible Gaussians {n_vis} of {st.N}")


@pytest.mark.parametrize("N,C,deg", [(1, 1, 3), (513, 3, 0), (1023, 2, 1), (70_001, 3, 2), (300_007, 4, 3)])
def test_grad_zero_rows_clears_exactly_the_union_of_the_mask(B, N, C, deg):
    """gs_grad_zero_rows against numpy: the rows of Gaussians marked in any view become zero, every other row (and nothing
    outside the arrays: they are allocated with a guard row on either side) keeps its contents; every SH degree, sizes
    around the 512-Gaussian mask granule and the 1024-Gaussian warp chunk."""
    rng = np.random.default_rng(N + deg)
    vis = rng.random((C, N)) < (0.5 if N < 2000 else 0.03)
    if N > 1:
        vis[:, N - 1] = [c == C - 1 for c in range(C)]           # the last Gaussian, in the last view only
    words = B.vis_words(N)
    mask = torch.from_numpy(pack_mask(vis, words)).cuda()
    K3 = 3 * (deg + 1) ** 2
    shapes = {"means": 3, "log_scales": 3, "quats": 4, "opacity_logits": 1, "sh": K3}
    full = {k: torch.full(((N + 2) * w,), 3.25, dtype=torch.float32, device="cuda") for k, w in shapes.items()}
    g = {k: full[k][shapes[k]: (N + 1) * shapes[k]].view(N, shapes[k]) if shapes[k] > 1 else full[k][1: N + 1] for k in shapes}
    # (the guard rows shift the alignment: unless the row width is a multiple of 4 floats the scalar store paths run here)
    B.gs_grad_zero_rows(deg, C, mask, g["means"], g["log_scales"], g["quats"], g["opacity_logits"], g["sh"])
    torch.cuda.synchronize()
    any_vis = torch.from_numpy(vis.any(axis=0)).cuda()
    for k, w in shapes.items():
        rows = g[k].reshape(N, -1)
        assert bool((rows[any_vis] == 0).all()), k
        assert bool((rows[~any_vis] == 3.25).all()), k
        assert bool((full[k][: w] == 3.25).all()) and bool((full[k][(N + 1) * w:] == 3.25).all()), k
    # aligned arrays take the 16-byte store paths: same result
    g2 = {k: torch.full((N, w) if w > 1 else (N,), 1.5, dtype=torch.float32, device="cuda") for k, w in shapes.items()}
    B.gs_grad_zero_rows(deg, C, mask, g2["means"], g2["log_scales"], g2["quats"], g2["opacity_logits"], g2["sh"])
    torch.cuda.synchronize()
    for k in shapes:
        rows = g2[k].reshape(N, -1)
        assert bool((rows[any_vis] == 0).all()) and bool((rows[~any_vis] == 1.5).all()), k
