"""-m gpu parity of the Davidson vector kernels (a8) against NumPy fp64 on the same inputs."""
import numpy as np
import pytest

import workloads as wlmod

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def ctx():
    from paper_2311_14106_b200 import dmrgk
    return dmrgk.Ctx(0)


def seeded(n, stream):
    return wlmod.normal12(77, stream, np.arange(n))


@pytest.mark.parametrize("n", [16, 48, 4096 + 16, 1 << 20])
@pytest.mark.parametrize("nv", [1, 3, 8, 17])
def test_multi_dot(ctx, n, nv):
    from paper_2311_14106_b200 import dmrgk
    X = seeded(n * nv, 1).reshape(nv, n)
    y = seeded(n, 2)
    Xd, yd = torch.from_numpy(X).cuda(), torch.from_numpy(y).cuda()
    out = torch.zeros(nv, dtype=torch.float64, device="cuda")
    scratch = torch.empty(dmrgk.vec_scratch_bytes(nv), dtype=torch.uint8, device="cuda")
    dmrgk.vec_multi_dot(ctx, n, nv, Xd, n, yd, out, scratch)
    ref = X @ y
    got = out.cpu().numpy()
    # error bound of a length-n dot: n·eps·Σ|x_i y_i| (pairwise in practice, far below)
    bound = 4 * np.finfo(float).eps * np.sqrt(n) * (np.abs(X) @ np.abs(y))
    assert np.all(np.abs(got - ref) <= bound)
    out2 = torch.zeros_like(out)
    dmrgk.vec_multi_dot(ctx, n, nv, Xd, n, yd, out2, scratch)
    assert torch.equal(out, out2)          # fixed-order reduction: bit-reproducible


@pytest.mark.parametrize("n", [16, 4096 + 32, 1 << 19])
def test_axpy_family(ctx, n):
    from paper_2311_14106_b200 import dmrgk
    nv = 5
    X = seeded(n * nv, 3).reshape(nv, n)
    y = seeded(n, 4)
    c = seeded(nv, 5)
    Xd, cd = torch.from_numpy(X).cuda(), torch.from_numpy(c).cuda()
    yd = torch.from_numpy(y).cuda()
    dmrgk.vec_multi_axpy(ctx, n, nv, Xd, n, cd, -1.0, 1.0, yd)
    ref = y - c @ X
    assert np.abs(yd.cpu().numpy() - ref).max() <= 1e-14 * np.abs(ref).max() * nv
    yd = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
    dmrgk.vec_multi_axpy(ctx, n, nv, Xd, n, cd, 1.0, 0.0, yd)      # beta = 0 never reads y
    assert np.abs(yd.cpu().numpy() - c @ X).max() <= 1e-14 * np.abs(ref).max() * nv
    xd, yd = torch.from_numpy(X[0]).cuda(), torch.from_numpy(y).cuda()
    dmrgk.vec_axpby(ctx, n, 0.25, xd, -3.0, yd)
    assert np.abs(yd.cpu().numpy() - (0.25 * X[0] - 3.0 * y)).max() <= 1e-15 * 8
    a = torch.tensor([7.5], dtype=torch.float64, device="cuda")
    for mode, f in ((0, 7.5), (1, 1 / 7.5), (2, np.sqrt(7.5)), (3, 1 / np.sqrt(7.5))):
        out = torch.empty(n, dtype=torch.float64, device="cuda")
        dmrgk.vec_scal_dev(ctx, n, a, mode, xd, out)
        assert np.abs(out.cpu().numpy() - f * X[0]).max() <= 1e-15 * 8


def test_residual_and_precond(ctx):
    from paper_2311_14106_b200 import dmrgk
    n, m = 4096 + 48, 6
    V = seeded(n * m, 6).reshape(m, n)
    W = seeded(n * m, 7).reshape(m, n)
    yv = seeded(m, 8)
    theta = -1.25
    coef = torch.from_numpy(np.concatenate([yv, [theta]])).cuda()
    r = torch.empty(n, dtype=torch.float64, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    scratch = torch.empty(dmrgk.vec_scratch_bytes(1), dtype=torch.uint8, device="cuda")
    dmrgk.vec_residual(ctx, n, m, torch.from_numpy(V).cuda(), torch.from_numpy(W).cuda(), n, coef, r, out, scratch)
    ref = yv @ W - theta * (yv @ V)
    assert np.abs(r.cpu().numpy() - ref).max() <= 1e-14 * np.abs(ref).max() * m
    assert abs(out.item() - ref @ ref) <= 1e-13 * (ref @ ref)
    d = seeded(n, 9)
    d[5] = theta                   # exact zero denominator → +1e-10
    d[6] = theta + 1e-12           # tiny negative denominator → −1e-10
    t = torch.empty(n, dtype=torch.float64, device="cuda")
    dmrgk.vec_precond(ctx, n, r, torch.from_numpy(d).cuda(), coef[m:], t)
    den = theta - d
    den = np.where(np.abs(den) < 1e-10, np.where(den < 0, -1e-10, 1e-10), den)
    rr = r.cpu().numpy()
    assert np.abs(t.cpu().numpy() - rr / den).max() <= 1e-15 * np.abs(rr / den).max() * 4


def test_blas1_names():
    """dmrgk_vec_dot / nrm2 / axpy / scal against NumPy."""
    from paper_2311_14106_b200 import dmrgk
    ctx = dmrgk.Ctx(0)
    n = 100_016
    rng = np.random.default_rng(3)
    xh, yh = rng.normal(size=n), rng.normal(size=n)
    x, y = torch.from_numpy(xh).cuda(), torch.from_numpy(yh).cuda()
    out = torch.zeros(8, dtype=torch.float64, device="cuda")
    scratch = torch.empty(dmrgk.vec_scratch_bytes(1), dtype=torch.uint8, device="cuda")
    dmrgk.vec_dot(ctx, n, x, y, out, scratch)
    assert abs(float(out[0]) - float(xh @ yh)) <= 1e-12 * np.linalg.norm(xh) * np.linalg.norm(yh)
    dmrgk.vec_nrm2(ctx, n, x, out, scratch)
    assert abs(float(out[0]) - np.linalg.norm(xh)) <= 1e-12 * np.linalg.norm(xh)
    dmrgk.vec_axpy(ctx, n, -0.75, x, y)
    assert np.array_equal(y.cpu().numpy(), np.asarray([-0.75 * a + b for a, b in zip(xh, yh)])) or \
        np.abs(y.cpu().numpy() - (-0.75 * xh + yh)).max() <= 1e-15 * np.abs(yh).max()
    dmrgk.vec_scal(ctx, n, 3.0, x)
    assert np.array_equal(x.cpu().numpy(), 3.0 * xh)
