"""gs_sort_pairs_static: the stand-alone radix sort with its scratch in a static device array (no workspace argument,
nothing allocated; include/gsplat_b200.h) against the existing path, gs_sort_pairs with a caller-owned workspace.
Integer work: bit for bit.  The file is named so that pytest collects it last (the suite runs with `pytest -x`).
It must pass alone in a fresh process and after the other GPU tests: it assumes nothing about what an earlier call
left in the shared scratch array, and checks that two calls in a row both come out right."""
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


def make_pairs(n, end_bit, skip, seed):
    rng = np.random.default_rng(seed)
    keys = rng.integers(0, 2 ** 63, n, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, n, dtype=np.uint64)
    mask = np.uint64((1 << end_bit) - 1 if end_bit < 64 else 0xFFFFFFFFFFFFFFFF)
    if skip:
        mask &= ~np.uint64(1 << 31)
    keys &= mask
    if n > 1000:
        keys[rng.integers(0, n, n // 3)] = keys[rng.integers(0, n, n // 3)]      # duplicates: stability matters
    return keys, np.arange(n, dtype=np.int32)


def sort_existing(B, keys, vals, end_bit, skip):
    n = len(keys)
    ws = torch.empty((B.gs_sort_pairs_workspace_bytes(n),), dtype=torch.uint8, device="cuda")
    dk, dv = torch.from_numpy(keys.view(np.int64)).cuda(), torch.from_numpy(vals).cuda()
    B.gs_sort_pairs(n, end_bit, skip, dk, dv, ws)
    torch.cuda.synchronize()
    return dk.cpu().numpy().view(np.uint64), dv.cpu().numpy()


def test_static_scratch_sort_equals_workspace_sort_on_two_calls_in_a_row(B):
    """Two calls in a row on one stream, different sizes / bit ranges / pass counts (the second one smaller, so a stale
    ticket, histogram or status word of the first call would be read), each against gs_sort_pairs and numpy's stable sort."""
    cases = [(B.GS_SORT_STATIC_MAX_N, 64, 0, 11), (300_001, 47, 1, 12), (4097, 33, 1, 13), (1, 64, 0, 14)]
    inputs = [make_pairs(n, e, s, seed) for n, e, s, seed in cases]
    dev = [(torch.from_numpy(k.view(np.int64)).cuda(), torch.from_numpy(v).cuda()) for k, v in inputs]
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for (n, e, s, _), (dk, dv) in zip(cases, dev):          # back to back, no synchronisation in between
        B.gs_sort_pairs_static(n, e, s, dk, dv)
    assert torch.cuda.memory_allocated() == before
    torch.cuda.synchronize()
    for (n, e, s, _), (keys, vals), (dk, dv) in zip(cases, inputs, dev):
        rk, rv = sort_existing(B, keys, vals, e, s)
        np.testing.assert_array_equal(dk.cpu().numpy().view(np.uint64), rk)
        np.testing.assert_array_equal(dv.cpu().numpy(), rv)
        order = np.argsort(keys, kind="stable")
        np.testing.assert_array_equal(rk, keys[order])
        np.testing.assert_array_equal(rv, vals[order])


def test_static_scratch_sort_repeats_the_same_call(B):
    """The same input twice in a row: the second call starts from the scratch the first one left behind."""
    n, e, s = 123_457, 49, 1
    keys, vals = make_pairs(n, e, s, 21)
    rk, rv = sort_existing(B, keys, vals, e, s)
    for _ in range(2):
        dk, dv = torch.from_numpy(keys.view(np.int64)).cuda(), torch.from_numpy(vals).cuda()
        B.gs_sort_pairs_static(n, e, s, dk, dv)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(dk.cpu().numpy().view(np.uint64), rk)
        np.testing.assert_array_equal(dv.cpu().numpy(), rv)


def test_static_scratch_sort_rejects_sizes_beyond_its_maximum(B):
    n = B.GS_SORT_STATIC_MAX_N + 1
    dk = torch.zeros((n,), dtype=torch.int64, device="cuda")
    dv = torch.arange(n, dtype=torch.int32, device="cuda")
    with pytest.raises(B.GsError) as ei:
        B.gs_sort_pairs_static(n, 64, 0, dk, dv)
    assert ei.value.status == B.GS_ERR_UNSUPPORTED
    assert "GS_SORT_STATIC_MAX_N" in str(ei.value)
    torch.cuda.synchronize()
    assert int(dk.abs().sum()) == 0 and bool((dv == torch.arange(n, dtype=torch.int32, device="cuda")).all())   # nothing ran
    B.gs_sort_pairs_static(0, 64, 0, None, None)            # n == 0: the set-up call, nothing to sort
    with pytest.raises(B.GsError):
        B.gs_sort_pairs_static(-1, 64, 0, dk, dv)
    with pytest.raises(B.GsError):
        B.gs_sort_pairs_static(16, 65, 0, dk, dv)
