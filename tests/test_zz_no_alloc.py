"""-m gpu test of dmrgk_vec_multi_dot_noalloc, the one entry point that needs no device allocation.

Who it is for: users of the library that cannot hand it a scratch buffer — a sweep driver whose operator
arenas and staging ring already fill HBM, a host code that is given a fixed set of device buffers and has
no allocator of its own, or a step running beside the side-stream operator copies, which a cudaMalloc /
cudaFree would stall by synchronising the device.  Its partial sums live in a fixed 592 KiB array inside
libdmrgk.so (nv ≤ 64), shared by every call on that GPU.

This file is named so that pytest collects it last: with `-x` a failure here hides nothing after it.
It builds its own context and inputs, so it passes alone in a fresh process as well as after the others.
"""
import numpy as np
import pytest

import workloads as wlmod

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _case(seed, n, nv):
    X = wlmod.normal12(seed, 1, np.arange(n * nv)).reshape(nv, n)
    y = wlmod.normal12(seed, 2, np.arange(n))
    return X, y


def test_noalloc_matches_scratch_path_twice_in_a_row():
    """Two calls in a row on the shared array — the second with fewer vectors and a shorter length, so it
    runs over slots the first one left filled — each compared with dmrgk_vec_multi_dot (caller's scratch):
    same kernels in the same fixed order, so the results are bit-identical, and both stay inside the
    dot-product error bound test_gpu_vec.py uses against NumPy."""
    from paper_2311_14106_b200 import dmrgk
    ctx = dmrgk.Ctx(0)
    for seed, n, nv in ((91, (1 << 20) + 48, 17), (92, 4096 + 16, 3)):
        X, y = _case(seed, n, nv)
        Xd, yd = torch.from_numpy(X).cuda(), torch.from_numpy(y).cuda()
        want = torch.zeros(nv, dtype=torch.float64, device="cuda")
        scratch = torch.empty(dmrgk.vec_scratch_bytes(nv), dtype=torch.uint8, device="cuda")
        dmrgk.vec_multi_dot(ctx, n, nv, Xd, n, yd, want, scratch)
        got = torch.full((nv,), float("nan"), dtype=torch.float64, device="cuda")
        dmrgk.vec_multi_dot_noalloc(ctx, n, nv, Xd, n, yd, got)
        torch.cuda.synchronize()
        assert torch.equal(got, want)
        bound = 4 * np.finfo(float).eps * np.sqrt(n) * (np.abs(X) @ np.abs(y))
        assert np.all(np.abs(got.cpu().numpy() - X @ y) <= bound)


def test_noalloc_largest_size_and_rejection():
    """nv = 64 is the most the built-in array holds; nv = 65 is refused with a message, before any launch."""
    from paper_2311_14106_b200 import dmrgk
    ctx = dmrgk.Ctx(0)
    n, nv = 1 << 19, 64                       # 1184 CTAs: every row of the array in use
    X, y = _case(93, n, nv)
    Xd, yd = torch.from_numpy(X).cuda(), torch.from_numpy(y).cuda()
    want = torch.zeros(nv, dtype=torch.float64, device="cuda")
    scratch = torch.empty(dmrgk.vec_scratch_bytes(nv), dtype=torch.uint8, device="cuda")
    dmrgk.vec_multi_dot(ctx, n, nv, Xd, n, yd, want, scratch)
    got = torch.full((nv,), float("nan"), dtype=torch.float64, device="cuda")
    dmrgk.vec_multi_dot_noalloc(ctx, n, nv, Xd, n, yd, got)
    torch.cuda.synchronize()
    assert torch.equal(got, want)
    X65 = torch.zeros(65 * 16, dtype=torch.float64, device="cuda")
    out = torch.zeros(65, dtype=torch.float64, device="cuda")
    before = dmrgk.launch_count()
    with pytest.raises(dmrgk.DmrgkError) as e:
        dmrgk.vec_multi_dot_noalloc(ctx, 16, 65, X65, 16, X65[:16], out)
    assert e.value.status == dmrgk.EINVAL and "64" in str(e.value)
    assert dmrgk.launch_count() == before
