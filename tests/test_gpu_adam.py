"""GPU parity of the fused Adam step (gs_adam_step) against oracle/adam_oracle.py through the C ABI.
Tolerance: one fp32 update of O(10) operations per element -> 2e-6 relative to max(|p|, lr) per element (the oracle
computes in double from the same fp32 inputs)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_11390_b200 import binding
    binding.lib()
    return binding


def f32(x):
    """The hyper-parameters reach the kernel as fp32: the oracle is given the same rounded values (1 - 0.999f differs from
    1 - 0.999 by 5e-5 relative)."""
    return float(np.float32(x))


def close(got, ref, scale):
    return np.abs(got.astype(np.float64) - ref).max() <= 2e-6 * scale


@pytest.mark.parametrize("N,row", [(1, 1), (1000, 3), (4097, 4), (333, 48), (100_003, 1), (50_001, 48)])
def test_dense_steps(B, N, row):
    from oracle import adam_oracle as A
    rng = np.random.default_rng(N + row)
    p = rng.standard_normal((N, row)).astype(np.float32)
    m = np.zeros_like(p); v = np.zeros_like(p)
    dp, dm, dv = (torch.from_numpy(x.copy()).cuda() for x in (p, m, v))
    lr, b1, b2, eps = f32(1e-2), f32(0.9), f32(0.999), f32(1e-15)
    rp, rm, rv = p.astype(np.float64), m.astype(np.float64), v.astype(np.float64)
    for t in range(1, 4):
        g = (rng.standard_normal((N, row)) * 10.0 ** rng.integers(-4, 1)).astype(np.float32)
        B.gs_adam_step(dp, torch.from_numpy(g).cuda(), dm, dv, lr, b1, b2, eps, t)
        # oracle from the fp32 state the kernel started the step with
        rp, rm, rv = A.adam_step(rp, g, rm, rv, lr, b1, b2, eps, t)
        torch.cuda.synchronize()
        gp, gm, gv = dp.cpu().numpy(), dm.cpu().numpy(), dv.cpu().numpy()
        assert close(gp, rp, max(np.abs(rp).max(), lr)) and close(gm, rm, np.abs(rm).max()) and close(gv, rv, np.abs(rv).max())
        rp, rm, rv = gp.astype(np.float64), gm.astype(np.float64), gv.astype(np.float64)


def test_unaligned_arrays_take_the_scalar_path(B):
    from oracle import adam_oracle as A
    rng = np.random.default_rng(5)
    buf = [torch.from_numpy(rng.standard_normal(3001).astype(np.float32)).cuda() for _ in range(4)]
    p, g, m, v = (b[1:] .view(1000, 3) for b in buf)                       # 4-byte aligned only
    v.abs_()
    ref = A.adam_step(p.cpu().numpy(), g.cpu().numpy(), m.cpu().numpy(), v.cpu().numpy(), f32(1e-3), f32(0.9), f32(0.999), f32(1e-8), 7)
    B.gs_adam_step(p, g, m, v, 1e-3, 0.9, 0.999, 1e-8, 7)
    torch.cuda.synchronize()
    for got, r in zip((p, m, v), ref):
        assert close(got.cpu().numpy(), r, np.abs(r).max())


@pytest.mark.parametrize("N,row,C,frac", [(5000, 48, 3, 0.05), (70_001, 3, 1, 0.5), (64, 4, 2, 0.0), (1000, 1, 4, 1.0)])
def test_visible_only_rows(B, N, row, C, frac):
    from oracle import adam_oracle as A
    rng = np.random.default_rng(N + C)
    p, g, m = (rng.standard_normal((N, row)).astype(np.float32) for _ in range(3))
    v = np.abs(rng.standard_normal((N, row))).astype(np.float32)
    radii = np.where(rng.random((C, N)) < frac, rng.integers(1, 50, (C, N)), 0).astype(np.int32)
    vis = (radii > 0).any(axis=0)
    ref = A.adam_step(p, g, m, v, f32(2e-3), f32(0.9), f32(0.999), f32(1e-15), 5, visible=vis)
    dp, dg, dm, dv = (torch.from_numpy(x.copy()).cuda() for x in (p, g, m, v))
    B.gs_adam_step(dp, dg, dm, dv, 2e-3, 0.9, 0.999, 1e-15, 5, radii=torch.from_numpy(radii).cuda())
    torch.cuda.synchronize()
    for got, r, old in zip((dp, dm, dv), ref, (p, m, v)):
        got = got.cpu().numpy()
        assert np.array_equal(got[~vis], old[~vis])                        # untouched rows: bit-exact
        if vis.any():
            assert close(got[vis], r[vis], np.abs(r).max())


@pytest.mark.parametrize("N,C,frac", [(4000, 4, 0.03), (10_001, 3, 0.3), (130, 1, 1.0), (5000, 2, 0.0)])
def test_visible_only_multi_array_step(B, N, C, frac):
    """gs_adam_step_visible: the five Gaussian arrays in one launch, radii scanned once; N not a multiple of 4 included."""
    from oracle import adam_oracle as A
    rng = np.random.default_rng(N * 7 + C)
    rows = (3, 3, 4, 1, 48)
    P = [rng.standard_normal((N, r)).astype(np.float32) for r in rows]
    G = [rng.standard_normal((N, r)).astype(np.float32) for r in rows]
    Ms = [rng.standard_normal((N, r)).astype(np.float32) for r in rows]
    Vs = [np.abs(rng.standard_normal((N, r))).astype(np.float32) for r in rows]
    radii = np.where(rng.random((C, N)) < frac, rng.integers(1, 50, (C, N)), 0).astype(np.int32)
    vis = (radii > 0).any(axis=0)
    hp = (f32(2e-3), f32(0.9), f32(0.999), f32(1e-15))
    dev = lambda xs: [torch.from_numpy(x.copy()).cuda() for x in xs]
    dP, dG, dM, dV = dev(P), dev(G), dev(Ms), dev(Vs)
    B.gs_adam_step_visible(dP, dG, dM, dV, *hp, 4, torch.from_numpy(radii).cuda())
    torch.cuda.synchronize()
    for q in range(5):
        ref = A.adam_step(P[q], G[q], Ms[q], Vs[q], *hp, 4, visible=vis)
        for got, r, old in zip((dP[q], dM[q], dV[q]), ref, (P[q], Ms[q], Vs[q])):
            got = got.cpu().numpy()
            assert np.array_equal(got[~vis], old[~vis])
            if vis.any():
                assert close(got[vis], r[vis], np.abs(r).max())
