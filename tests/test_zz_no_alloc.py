"""uts_depth_order_static: the depth order (Alg.1 l.15 PAPER.md:560, moved ahead of the query) for callers that cannot allocate — the
scratch is a file-scope device array of the library (include/uts.h).  Its emit_rank must equal uts_depth_order's, bit for bit (the
bar of every integer stage), on two calls in a row that share the array: the second call is smaller and has other views, so stale
contents of the first would show.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

pytestmark = pytest.mark.gpu


def _gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_29794_b200 import binding as B
    return B


def _rho(n_views, n_gauss, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    rho = torch.rand(n_views, n_gauss, device="cuda", generator=g) * 40.0 + 0.5
    rho[:, ::7] = rho[:, 3:4]                          # heavy ties: the order among equal depths is by Gaussian id
    return rho.contiguous()


def test_static_scratch_depth_order_equals_the_caller_scratch_path_twice_in_a_row():
    B = _gpu()
    limit = B.uts_depth_order_static_max()
    assert limit == 262144
    for n_views, n_gauss, seed in ((1, limit, 1), (3, 50_001, 2)):         # the maximum size first, then a smaller, ragged, 3-view call
        cfg = B.Config(order=6, n_gauss=n_gauss, n_views=n_views)
        rho = _rho(n_views, n_gauss, seed)
        n = n_views * n_gauss
        want = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        scratch = torch.empty(B.uts_depth_order_scratch_bytes(cfg) // 8 + 32, dtype=torch.int64, device="cuda")
        B.uts_depth_order(cfg, rho, want, scratch)
        got = torch.full((n,), -2, dtype=torch.int32, device="cuda")
        B.uts_depth_order_static(cfg, rho, got)
        torch.cuda.synchronize()
        assert torch.equal(got, want)
        # and it is the order it claims to be: a permutation whose inverse sorts by (view, depth bits, id)
        order = torch.empty_like(got, dtype=torch.int64)
        order[got.long()] = torch.arange(n, device="cuda")
        key = (order // n_gauss) * (1 << 32) + rho.view(-1)[order].view(torch.int32).long()
        assert bool((key[1:] >= key[:-1]).all())
        tie = key[1:] == key[:-1]
        assert bool((order[1:][tie] > order[:-1][tie]).all())


def test_static_scratch_refuses_sizes_beyond_its_limit():
    B = _gpu()
    limit = B.uts_depth_order_static_max()
    cfg = B.Config(order=6, n_gauss=limit // 2 + 1, n_views=2)
    rho = torch.ones(2, limit // 2 + 1, device="cuda")
    out = torch.full((2 * (limit // 2 + 1),), 5, dtype=torch.int32, device="cuda")
    with pytest.raises(B.UtsError) as ei:
        B.uts_depth_order_static(cfg, rho, out)
    assert ei.value.status == B.UTS_ERR_CAPACITY and str(limit) in str(ei.value)
    torch.cuda.synchronize()
    assert int((out != 5).sum()) == 0                  # nothing was enqueued
    B.uts_depth_order_static(B.Config(order=6, n_gauss=0), rho, out)       # empty input: no work, no error
