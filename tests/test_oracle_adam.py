"""Pins of the Adam oracle: torch.optim.Adam (a library routine) over several steps, a hand-computed first step, and the
visible-only variant's defining property."""
import numpy as np
import torch

from oracle import adam_oracle as A


def test_matches_torch_optim_adam_over_several_steps():
    rng = np.random.default_rng(0)
    p0 = rng.standard_normal((50, 7))
    grads = [rng.standard_normal((50, 7)) * (0.1 + k) for k in range(6)]
    lr, b1, b2, eps = 1.6e-3, 0.9, 0.999, 1e-15
    tp = torch.tensor(p0, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([tp], lr=lr, betas=(b1, b2), eps=eps)
    p, m, v = p0.copy(), np.zeros_like(p0), np.zeros_like(p0)
    for t, g in enumerate(grads, start=1):
        tp.grad = torch.tensor(g, dtype=torch.float64)
        opt.step()
        p, m, v = A.adam_step(p, g, m, v, lr, b1, b2, eps, t)
        assert np.abs(p - tp.detach().numpy()).max() <= 1e-13
    st = opt.state[tp]
    assert np.abs(m - st["exp_avg"].numpy()).max() <= 1e-14 and np.abs(v - st["exp_avg_sq"].numpy()).max() <= 1e-14


def test_first_step_closed_form():
    # t = 1, m = v = 0: m_hat = g, v_hat = g^2 -> p - lr g / (|g| + eps) = p - lr sign(g) (for |g| >> eps)
    p, m, v = A.adam_step(np.array([1.0, -2.0]), np.array([0.5, -4.0]), np.zeros(2), np.zeros(2), 0.01, 0.9, 0.999, 1e-30, 1)
    assert np.allclose(p, [0.99, -1.99], rtol=0, atol=1e-15)
    assert np.allclose(m, [0.05, -0.4]) and np.allclose(v, [0.00025, 0.016])


def test_visible_only_rows():
    rng = np.random.default_rng(1)
    p, g, m, v = (rng.standard_normal((20, 3)) for _ in range(4))
    v = np.abs(v)
    vis = rng.random(20) < 0.4
    pd, md, vd = A.adam_step(p, g, m, v, 1e-2, 0.9, 0.999, 1e-8, 3)
    ps, ms, vs = A.adam_step(p, g, m, v, 1e-2, 0.9, 0.999, 1e-8, 3, visible=vis)
    assert np.array_equal(ps[vis], pd[vis]) and np.array_equal(ms[vis], md[vis]) and np.array_equal(vs[vis], vd[vis])
    assert np.array_equal(ps[~vis], p[~vis]) and np.array_equal(ms[~vis], m[~vis]) and np.array_equal(vs[~vis], v[~vis])
