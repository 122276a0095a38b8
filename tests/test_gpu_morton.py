"""GPU parity of the Morton ordering (gs_bounds, gs_morton_codes, gs_sort_pairs, gs_gather_rows)
against oracle/morton_oracle.py through the C ABI.  Integer work: everything is compared bit for bit."""
import numpy as np
import pytest

from paper_2606_11390_b200 import scenes

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_11390_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def oracle():
    from oracle import morton_oracle
    return morton_oracle


def gpu_codes(B, means):
    d = torch.from_numpy(means).cuda()
    lo_hi = torch.empty((6,), dtype=torch.float32, device="cuda")
    codes = torch.empty((means.shape[0],), dtype=torch.int64, device="cuda")
    index = torch.empty((means.shape[0],), dtype=torch.int32, device="cuda")
    B.gs_bounds(d, lo_hi)
    B.gs_morton_codes(d, lo_hi, codes, index)
    torch.cuda.synchronize()
    return lo_hi.cpu().numpy(), codes.cpu().numpy().view(np.uint64), index.cpu().numpy()


@pytest.mark.parametrize("name,n", [("tiny", None), ("object", 100_003), ("block", 300_001), ("city", 1_000_000)])
def test_bounds_and_codes_bit_exact(B, oracle, name, n):
    means = scenes.make_scene(name, n=n)["means"]
    lo, hi = oracle.bounds(means)
    lo_hi, codes, index = gpu_codes(B, means)
    assert np.array_equal(lo_hi[:3], lo) and np.array_equal(lo_hi[3:], hi)
    assert np.array_equal(codes, oracle.morton_codes(means, lo, hi))
    assert np.array_equal(index, np.arange(means.shape[0], dtype=np.int32))


def test_degenerate_axes_negative_and_nonfinite_values(B, oracle):
    rng = np.random.default_rng(0)
    means = rng.uniform(-5, -1, (1000, 3)).astype(np.float32)
    means[:, 2] = -3.25                                    # degenerate axis, negative coordinates
    lo_hi, codes, _ = gpu_codes(B, means)
    lo, hi = oracle.bounds(means)
    assert np.array_equal(lo_hi[:3], lo) and np.array_equal(lo_hi[3:], hi)
    assert np.array_equal(codes, oracle.morton_codes(means, lo, hi))
    one = np.array([[1.5, -2.0, 7.0]], np.float32)         # a single Gaussian: every axis degenerate, code 0
    lo_hi, codes, _ = gpu_codes(B, one)
    assert codes.tolist() == [0] and lo_hi.tolist() == [1.5, -2.0, 7.0, 1.5, -2.0, 7.0]


def test_morton_sort_of_all_parameter_arrays(B, oracle):
    sc = scenes.make_scene("object", n=50_007)
    names = ("means", "log_scales", "quats", "opacity_logits", "sh")
    params = {k: torch.from_numpy(np.ascontiguousarray(sc[k], dtype=np.float32)).cuda() for k in names}
    out, perm = B.morton_sort(params)
    torch.cuda.synchronize()
    want = oracle.morton_order(sc["means"])
    assert np.array_equal(perm.cpu().numpy(), want)        # stable: ties in ascending index
    for k in names:
        assert np.array_equal(out[k].cpu().numpy(), np.asarray(sc[k], np.float32)[want]), k


def test_sorted_scene_renders_the_same_image(B):
    """Permuting the Gaussians leaves the image unchanged up to the order of equal-depth records (none here)."""
    from paper_2606_11390_b200.pipeline import SplatStep
    sc = scenes.make_scene("tiny")
    ref = SplatStep(sc)
    ref.forward(sync=True)
    params = {k: ref.params[k] for k in ref.param_names}
    out, perm = B.morton_sort(params)
    st = SplatStep(sc)
    for k in st.param_names:
        st.params[k].copy_(out[k])
    st.forward(sync=True)
    torch.cuda.synchronize()
    assert st.M == ref.M
    assert torch.equal(st.n_contrib, ref.n_contrib)
    assert float((st.image - ref.image).abs().max()) <= 1e-6
