"""cos_eval_connected_noalloc (include/cos.h): the allocation-free entry point against the existing path.

Collected last on purpose (the suite runs with `pytest -x`): a failure here hides nothing after it.  The entry point
keeps the pair kernel's records and item descriptors in a static device array shared by every call on the GPU, so the
checks are: (1) two calls in a row -- different orders, species counts and inputs, so the second call finds the array
full of the first one's records and descriptors -- each agree with cos_eval_connected on the same inputs; (2) a repeat
of a call returns the same bits; (3) sizes beyond the stated maximum are refused with COS_ETOOBIG and nothing else runs.

Tolerance: rtol 1e-10, the one tests/test_gpu_parity.py uses between two evaluations whose team sizes may differ
(cos.h, determinism note); inputs are the well-conditioned random matrices of that test."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

RTOL = 1e-10


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device: the CUDA path has no CPU fallback")
    from paper_2501_00675_b200 import build
    build.build()
    return torch


@pytest.fixture(scope="module")
def ctx(torch_mod):
    from paper_2501_00675_b200 import api
    c = api.Context()
    yield c
    c.close()


def _inputs(torch, seed, n, nsp, B):
    rng = np.random.default_rng(seed)
    Gup = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)
    Gdn = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n) if nsp == 2 else None
    u = rng.uniform(0.5, 2.0, size=(B, n))
    dGup = torch.from_numpy(Gup).cuda()
    dGdn = dGup if Gdn is None else torch.from_numpy(Gdn).cuda()
    return dGup, dGdn, torch.from_numpy(u).cuda()


def _run(torch, fn, dGup, dGdn, du, U):
    out = torch.full((dGup.shape[0],), float("nan"), dtype=torch.float64, device="cuda")
    fn(dGup, dGdn, out, U=U, d_u=du)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def test_noalloc_matches_existing_path_on_consecutive_calls(torch_mod, ctx):
    torch = torch_mod
    # consecutive calls through the static array; sizes span one partial grid round, several rounds and a ragged tail
    calls = [(12, 2, 700), (11, 1, 2500), (12, 1, 1201), (11, 2, 333), (12, 1, 5)]
    prepared = [(n, nsp, B) + _inputs(torch, 9100 + i, n, nsp, B) for i, (n, nsp, B) in enumerate(calls)]
    # the static-scratch calls run back to back, nothing of the existing path in between
    got = [_run(torch, ctx.eval_connected_noalloc, gu, gd, u, 1.3) for (_, _, _, gu, gd, u) in prepared]
    assert ctx.last_kernel_name().startswith("eval_pair_kernel")
    for (n, nsp, B, gu, gd, u), g in zip(prepared, got):
        ref = _run(torch, ctx.eval_connected, gu, gd, u, 1.3)
        assert np.all(np.isfinite(g)) and g.shape == (B,)
        np.testing.assert_allclose(g, ref, rtol=RTOL, err_msg=f"n={n} nsp={nsp} batch={B}")
    # after the existing path ran (its own scratch, another order of descriptors): same bits as before
    for (n, nsp, B, gu, gd, u), g in zip(prepared, got):
        np.testing.assert_array_equal(_run(torch, ctx.eval_connected_noalloc, gu, gd, u, 1.3), g)


def test_noalloc_second_context_and_empty_batch(torch_mod, ctx):
    """Another context on the same GPU resolves the same array; batch 0 is legal and launches nothing."""
    torch = torch_mod
    from paper_2501_00675_b200 import api
    gu, gd, u = _inputs(torch, 9200, 11, 2, 64)
    a = _run(torch, ctx.eval_connected_noalloc, gu, gd, u, 0.7)
    with api.Context() as other:
        b = _run(torch, other.eval_connected_noalloc, gu, gd, u, 0.7)
        e = torch.empty((0, 11, 11), dtype=torch.float64, device="cuda")
        other.eval_connected_noalloc(e, e, torch.empty((0,), dtype=torch.float64, device="cuda"),
                                     d_u=torch.empty((0, 11), dtype=torch.float64, device="cuda"))
        assert other.last_launch_count() == 0
    np.testing.assert_array_equal(a, b)
    np.testing.assert_allclose(a, _run(torch, ctx.eval_connected, gu, gd, u, 0.7), rtol=RTOL)


def test_noalloc_rejects_sizes_beyond_the_maximum(torch_mod, ctx):
    torch = torch_mod
    from paper_2501_00675_b200 import api
    for n, code in [(13, api.COS_ETOOBIG), (16, api.COS_ETOOBIG), (10, api.COS_EINVAL), (4, api.COS_EINVAL)]:
        gu, gd, u = _inputs(torch, 9300 + n, n, 1, 8)
        out = torch.full((8,), 7.0, dtype=torch.float64, device="cuda")
        with pytest.raises(api.CosError) as ei:
            ctx.eval_connected_noalloc(gu, gd, out, d_u=u)
        assert ei.value.code == code
        torch.cuda.synchronize()
        assert bool((out == 7.0).all())           # a refused call writes nothing
    assert "capacity" in api.strerror(api.COS_ETOOBIG)
    # batch above COS_NOALLOC_MAX_BATCH: refused on the sizes alone (the pointers are never dereferenced)
    lib = api.load_library()
    one = torch.zeros(1, dtype=torch.float64, device="cuda")
    rc = lib.cos_eval_connected_noalloc(ctx._h, 11, api.COS_NOALLOC_MAX_BATCH + 1, one.data_ptr(), one.data_ptr(), None,
                                        1.0, one.data_ptr())
    assert rc == api.COS_ETOOBIG
