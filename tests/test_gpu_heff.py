"""-m gpu parity: σ = H_eff ψ from the CUDA library (through the C ABI) against the oracle,
element by element on the same seeded inputs (BASELINE.json: relative max-norm ≤ 1e-11)."""
import numpy as np
import pytest

import workloads as wlmod
from oracle import heff, lattice, dmrg, export
from _gpu import device_problem, rel_max, padding_is_zero, config1_problem, TOL_SIGMA

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def small_config2():
    return wlmod.synthetic_config2(M=64, n_q=9, K=32, seed=2, width2=8.0)


def medium_config2():
    # several 64×64 tiles per block, ragged tails (sector sizes 1 … 100), split-k exercised
    return wlmod.synthetic_config2(M=400, n_q=13, K=40, seed=12, width2=10.0)


def small_spinless():
    return wlmod.lattice_workload("spinless", 5, 24, seed=3)


def medium_spinless():
    thin = lambda fam, i: fam in ("F1", "F2") or i % 5 == 0
    return wlmod.lattice_workload("spinless", 10, 600, seed=13, width2=4.0, keep=thin)


def small_hubbard():
    thin = lambda fam, i: fam in ("F1", "F2") or i % 3 == 0
    return wlmod.lattice_workload("hubbard", 2, 14, seed=4, keep=thin)


def medium_hubbard():
    thin = lambda fam, i: fam in ("F1", "F2") or i % 7 == 0
    return wlmod.lattice_workload("hubbard", 5, 400, seed=14, keep=thin)


@pytest.mark.parametrize("make", [small_config2, small_spinless, small_hubbard])
@pytest.mark.parametrize("kernel", [0, 1])
def test_sigma_vs_dense_kronecker(make, kernel):
    """T2: H_eff assembled densely by explicit Kronecker products with Jordan–Wigner signs."""
    pb = heff.problem_from_workload(make())
    ref = heff.sigma_dense(pb)
    dp = device_problem(pb, kernel=kernel)
    psi = dp.psi_from_host(pb.psi)
    sigma = dp.apply(psi)
    assert rel_max(dp.to_blocks(sigma), ref) <= TOL_SIGMA
    assert padding_is_zero(dp, sigma)
    assert dp.heff.flops_alg == heff.flops_alg(pb)
    assert dp.heff.n_tasks == len(heff.enumerate_tasks(pb))


@pytest.mark.parametrize("make", [medium_config2, medium_spinless, medium_hubbard])
@pytest.mark.parametrize("opts", [{}, {"split_waves": 4}, {"t_chunk_bytes": 1 << 20}, {"order_policy": 1}, {"order_policy": 2},
                                  {"kernel": 4}, {"kernel": 4, "split_waves": 64}])
def test_sigma_vs_blockwise_medium(make, opts):
    """T3 at sizes spanning several tiles and ragged tails; split-k and chunking variants, and the
    tall-tile (128×64) variant of the GEMM kernel."""
    pb = heff.problem_from_workload(make())
    ref = heff.sigma_blockwise(pb)
    dp = device_problem(pb, **opts)
    sigma = dp.apply(dp.psi_from_host(pb.psi))
    assert rel_max(dp.to_blocks(sigma), ref) <= TOL_SIGMA
    assert padding_is_zero(dp, sigma)
    if "t_chunk_bytes" in opts:
        assert dp.heff.n_chunks > 1
    assert dp.heff.flops_alg == heff.flops_alg(pb)
    has_identity = any(L is None or R is None for (L, R, _, _, _) in pb.terms)
    if opts.get("order_policy", 0) == 0 and not has_identity:
        assert dp.heff.flops_exec == dp.heff.flops_alg        # every task in its cheaper order
    else:
        assert dp.heff.flops_exec >= dp.heff.flops_alg        # identity factors are executed as products


def test_gemm_order_is_chosen_per_task_on_skewed_shapes():
    """Sectors of very different sizes on the two halves: (Lψ)Rᵀ is cheaper for some tasks, L(ψRᵀ) for
    others.  All three policies give the oracle's σ; only the automatic one executes the
    algorithmic flop count; a staged (pinned) run goes through the same code with both orders present."""
    from paper_2311_14106_b200 import problem
    secA = [((q,), d) for q, d in enumerate([3, 70, 5, 130, 9, 2])]
    secB = [((q,), d) for q, d in enumerate([90, 4, 150, 6, 40, 11])]
    wl = wlmod.Workload("skewed", 21, 1, secA, secB, (5,))
    shifts = [1, -1, 2, 0, -2, 1, -1, 0]
    for k, dlt in enumerate(shifts):
        wl.ops.append(wlmod.OpSpec("A", (dlt,), dlt & 1, False, "one", f"L{k}"))
        wl.ops.append(wlmod.OpSpec("B", (-dlt,), dlt & 1, False, "one", f"R{k}"))
        wl.terms.append(wlmod.TermSpec(2 * k, 2 * k + 1, 0.3 + 0.1 * k, False, False, "syn"))
        wl.terms.append(wlmod.TermSpec(2 * k, 2 * k + 1, -0.2 + 0.05 * k, True, True, "syn^T"))
    pb = heff.problem_from_workload(wl)
    ref = heff.sigma_blockwise(pb)
    execd = {}
    for policy in (0, 1, 2):
        dp = device_problem(pb, order_policy=policy)
        sigma = dp.apply(dp.psi_from_host(pb.psi))
        assert rel_max(dp.to_blocks(sigma), ref) <= TOL_SIGMA, policy
        assert padding_is_zero(dp, sigma)
        assert rel_max(dp.to_blocks(dp.diag()), heff.diagonal_blockwise(pb)) <= 1e-13
        execd[policy] = dp.heff.flops_exec
        assert dp.heff.flops_alg == heff.flops_alg(pb)
    assert execd[0] == heff.flops_alg(pb) and execd[1] > execd[0] and execd[2] > execd[0]     # both orders are in use
    for kern in (2, 3, 4):                                  # the other residencies and the tall tile, same lists
        dp = device_problem(pb, kernel=kern)
        sigma = dp.apply(dp.psi_from_host(pb.psi))
        assert rel_max(dp.to_blocks(sigma), ref) <= TOL_SIGMA, kern
        assert padding_is_zero(dp, sigma)
    stg = problem.from_workload(wl, pinned=[1, 2, 6, 9], ring_bytes=64 << 20)
    got = stg.apply(stg.psi_fill(wl.seed, wlmod.PSI_STREAM))
    res = problem.from_workload(wl)
    want = res.apply(res.psi_fill(wl.seed, wlmod.PSI_STREAM))
    torch.cuda.synchronize()
    assert torch.equal(got, want)


def test_device_fill_matches_host_generator():
    """The library's seeded fill kernel reproduces workloads.fill_op_host bit for bit, so
    device-generated arenas and the oracle's host blocks are the same inputs."""
    from paper_2311_14106_b200 import problem
    for wl in (small_config2(), small_spinless(), small_hubbard()):
        dp = problem.from_workload(wl)
        for i in range(len(wl.ops)):
            host = wlmod.fill_op_host(wl, i)
            dev = dp.read_op_blocks(i)
            assert set(host) == set(dev)
            for k in host:
                assert np.array_equal(host[k], dev[k]), (wl.name, i, k)
        psi = dp.to_blocks(dp.psi_fill(wl.seed, wlmod.PSI_STREAM))
        ref = wlmod.fill_psi_host(wl)
        for k in ref:
            assert np.array_equal(psi[k], ref[k])


def test_config2_full_size():
    """BASELINE.json configs[1] (M=1024, 33 sectors, K=512) against T3, all blocks."""
    from paper_2311_14106_b200 import problem
    wl = wlmod.synthetic_config2()
    pb = heff.problem_from_workload(wl)
    ref = heff.sigma_blockwise(pb)
    dp = problem.from_workload(wl)
    sigma = dp.apply(dp.psi_fill(wl.seed, wlmod.PSI_STREAM))
    assert rel_max(dp.to_blocks(sigma), ref) <= TOL_SIGMA
    assert dp.heff.flops_alg == heff.flops_alg(pb)


@pytest.fixture(scope="module")
def config1():
    return config1_problem()


def test_config1_sigma_vs_definition_and_kronecker(config1):
    """σ_gpu vs P†HP ψ (T1, the definition) and vs the dense Kronecker H_eff (T2)."""
    pb, Heff, x, space = config1
    dp = device_problem(pb)
    sigma = dp.to_blocks(dp.apply(dp.psi_from_host(pb.psi)))
    ref1 = dmrg.vec_to_blocks(space, Heff @ x)
    assert rel_max(sigma, ref1) <= TOL_SIGMA
    assert rel_max(sigma, heff.sigma_dense(pb)) <= TOL_SIGMA


def test_hermiticity_and_linearity():
    """⟨x, Hy⟩ = ⟨Hx, y⟩ pins the h.c. pairing and the fermionic sign rule; σ is linear in ψ."""
    from paper_2311_14106_b200 import problem
    wl = medium_hubbard()
    dp = problem.from_workload(wl)
    n = dp.layout.n_padded
    x = dp.psi_fill(wl.seed, 101)
    y = dp.psi_fill(wl.seed, 102)
    Hx, Hy = dp.apply(x), dp.apply(y)
    a, b = torch.dot(x[:n], Hy[:n]).item(), torch.dot(Hx[:n], y[:n]).item()
    scale = torch.linalg.norm(Hx[:n]).item() * torch.linalg.norm(y[:n]).item()
    assert abs(a - b) <= 1e-12 * scale
    z = (0.3 * x - 1.7 * y).contiguous()
    Hz = dp.apply(z)
    ref = 0.3 * Hx - 1.7 * Hy
    assert (Hz - ref).abs().max().item() <= 1e-12 * ref.abs().max().item()


def test_block_support_single_block_input():
    """ψ supported on one block reaches only blocks shifted by some δ_k (charge conservation)."""
    wl = small_spinless()
    pb = heff.problem_from_workload(wl)
    keys = pb.psi_blocks()
    mid = keys[len(keys) // 2]
    psi = {k: (v if k == mid else np.zeros_like(v)) for k, v in pb.psi.items()}
    ref = heff.sigma_blockwise(pb, psi)
    dp = device_problem(pb)
    got = dp.to_blocks(dp.apply(dp.psi_from_host(psi)))
    assert rel_max(got, ref) <= TOL_SIGMA
    for k in ref:
        if not np.any(ref[k]):
            assert not np.any(got[k])


def test_k_additivity():
    """σ(K list) = σ(first half) + σ(second half)."""
    pb = heff.problem_from_workload(medium_config2())
    dp = device_problem(pb)
    psi = dp.psi_from_host(pb.psi)
    full = dp.apply(psi).clone()
    K = len(pb.terms)
    parts = []
    for sl in (slice(0, K // 2), slice(K // 2, K)):
        dp.build(pb.terms[sl])
        parts.append(dp.apply(psi).clone())
    s = parts[0] + parts[1]
    assert (full - s).abs().max().item() <= 1e-12 * full.abs().max().item()


def test_diag_matches_oracle():
    for make in (small_config2, medium_spinless, small_hubbard):
        pb = heff.problem_from_workload(make())
        dp = device_problem(pb)
        got = dp.to_blocks(dp.diag())
        ref = heff.diagonal_blockwise(pb)
        assert rel_max(got, ref) <= 1e-13


def test_staged_operators_bit_identical_to_resident():
    """a3: operators streamed from pinned host memory through the ring.  With the same chunk
    boundaries (ring large enough that only t_chunk_bytes cuts the pair list) the staged run gives
    the same bits as the resident one; with a small ring (more chunks, a different summation order
    over chunks) it agrees to rounding and is reproducible call after call."""
    from paper_2311_14106_b200 import problem
    wl = medium_spinless()
    res = problem.from_workload(wl, t_chunk_bytes=1 << 20)
    psi = res.psi_fill(wl.seed, wlmod.PSI_STREAM)
    ref = res.apply(psi).clone()
    pinned = [i for i in range(len(wl.ops)) if i % 3 == 1]
    stg = problem.from_workload(wl, pinned=pinned, ring_bytes=256 << 20, t_chunk_bytes=1 << 20)
    assert stg.heff.n_chunks == res.heff.n_chunks > 2
    for _ in range(2):      # second call re-uses the ring parts
        got = stg.apply(stg.psi_fill(wl.seed, wlmod.PSI_STREAM))
        torch.cuda.synchronize()
        assert torch.equal(got, ref)
    assert torch.equal(stg.diag(), res.diag())
    small = problem.from_workload(wl, pinned=pinned, ring_bytes=2000000, t_chunk_bytes=1 << 20)
    assert small.heff.n_chunks >= res.heff.n_chunks
    first = small.apply(psi).clone()
    again = small.apply(psi)
    torch.cuda.synchronize()
    assert torch.equal(first, again)
    assert float((first - ref).abs().max() / ref.abs().max()) <= 1e-13


def test_staging_ring_too_small_for_a_pair_is_refused():
    """Both operators of a pair are staged into the same ring part: a ring whose third holds either
    operator alone but not the two together must be refused at create time (DMRGK_ENOMEM), not
    overflowed at apply time."""
    from paper_2311_14106_b200 import dmrgk, problem
    wl = medium_spinless()
    probe = problem.from_workload(wl)
    pairs = [(t.L, t.R) for t in wl.terms if t.L is not None and t.R is not None]
    L, R = max(pairs, key=lambda p: probe.ops[p[0]].n_padded + probe.ops[p[1]].n_padded)
    nl, nr = probe.ops[L].n_padded * 8, probe.ops[R].n_padded * 8
    third = (max(nl, nr) + nl + nr) // 2 // 128 * 128          # ≥ each alone, < both together
    assert max(nl, nr) <= third < nl + nr
    with pytest.raises(dmrgk.DmrgkError) as e:
        problem.from_workload(wl, pinned=[L, R], ring_bytes=3 * third)
    assert e.value.status == dmrgk.ENOMEM
    ok = problem.from_workload(wl, pinned=[L, R], ring_bytes=3 * (nl + nr + 256))
    psi = ok.psi_fill(wl.seed, wlmod.PSI_STREAM)
    ref = probe.apply(probe.psi_fill(wl.seed, wlmod.PSI_STREAM))
    got = ok.apply(psi)
    torch.cuda.synchronize()
    assert float((got - ref).abs().max() / ref.abs().max()) <= 1e-13


def test_hc_of_prev_flag_equals_explicit_transposes():
    """DMRGK_HC_OF_PREV: 'pair k is the h.c. of pair k−1' gives the same bits as naming the same stored
    operators with both transpose flags (SURVEY §8(b) flag list)."""
    pb = heff.problem_from_workload(medium_spinless())
    explicit = device_problem(pb)
    terms = []
    for k, (L, R, c, tL, tR) in enumerate(pb.terms):
        prev = pb.terms[k - 1] if k else None
        if prev is not None and tL and tR and (L, R) == (prev[0], prev[1]) and not prev[3] and not prev[4]:
            terms.append((None, None, c, "hc", "hc"))
        else:
            terms.append((L, R, c, tL, tR))
    assert any(t[3] == "hc" for t in terms)
    from paper_2311_14106_b200 import problem
    dp = problem.from_host(pb.n_charges, pb.sectors_A, pb.sectors_B, pb.target, pb.ops, terms)
    a = explicit.apply(explicit.psi_from_host(pb.psi))
    b = dp.apply(dp.psi_from_host(pb.psi))
    torch.cuda.synchronize()
    assert torch.equal(a, b) and dp.heff.n_tasks == explicit.heff.n_tasks


def test_apply_host_end_to_end():
    wl = medium_config2()
    pb = heff.problem_from_workload(wl)
    dp = device_problem(pb)
    psi_dev = dp.psi_from_host(pb.psi)
    ref = dp.apply(psi_dev).clone()
    n = dp.layout.n_padded
    ph = psi_dev[:n].cpu().pin_memory()
    sh = torch.empty(n, dtype=torch.float64).pin_memory()
    dp.heff.apply_host(ph, sh, dp.new_vector(), dp.new_vector(), dp.workspace, dp.stream, dp.copy_stream)
    assert torch.equal(sh, ref[:n].cpu())


def test_edge_cases_and_errors():
    from paper_2311_14106_b200 import dmrgk, problem
    sec = [((q,), d) for q, d in enumerate([1, 3, 0, 17, 2])]
    # K = 0: σ = 0
    dp = problem.DeviceProblem(1, sec, sec, (4,))
    dp.create_ops([])
    dp.build([])
    sigma = dp.apply(dp.psi_fill(1, 7))
    assert dp.heff.n_tasks == 0 and not torch.any(sigma)
    # no allowed block: apply is a no-op, Davidson refuses
    empty = problem.DeviceProblem(1, sec, sec, (99,))
    assert empty.layout.n_blocks == 0
    empty.create_ops([])
    empty.build([])
    empty.apply(empty.new_vector())
    # shifts that do not cancel / parity mismatch / wrong space / unbound
    dp.create_ops([("A", (1,), 1), ("B", (1,), 1), ("B", (-1,), 0), ("A", (-1,), 1)])
    dp.alloc_resident()
    for terms, code in (([(0, 1, 1.0, False, False)], dmrgk.ECHARGE),
                        ([(0, 2, 1.0, False, False)], dmrgk.ECHARGE),
                        ([(0, 3, 1.0, False, False)], dmrgk.ESHAPE)):
        with pytest.raises(dmrgk.DmrgkError) as e:
            dp.build(terms)
        assert e.value.status == code
    dp.build([(0, 1, 1.0, False, True)])        # transposing R makes the shifts cancel
    unb = dmrgk.Op(dp.ctx, dp.A, (1,), 1)
    with pytest.raises(dmrgk.DmrgkError) as e:
        dmrgk.Heff(dp.ctx, dp.layout, [(unb, dp.ops[1], 1.0, False, True)])
    assert e.value.status == dmrgk.ESTATE
    # misaligned pointers
    v = dp.new_vector()
    with pytest.raises(dmrgk.DmrgkError) as e:
        dp.heff.apply(v.data_ptr() + 8, v, dp.workspace)
    assert e.value.status == dmrgk.EALIGN
    with pytest.raises(dmrgk.DmrgkError) as e:
        dp.heff.apply(v, v, dp.workspace)
    assert e.value.status == dmrgk.EINVAL


def test_block_coefficients_su2_slot():
    """dmrgk_heff_create_blockcoef: one extra scalar per (pair, input block) — the slot of the SU(2)
    recoupling coefficients — against the oracle with random scalars (zeros remove
    tasks), and the spin-singlet H_eff of the Hubbard dimer: σ and the Davidson energy against the
    closed form (U − √(U² + 16t²))/2."""
    from paper_2311_14106_b200 import problem
    from _su2 import dimer_singlet_problem
    from _util import golden_table

    def on_device(pb, **opts):
        dp = problem.DeviceProblem(pb.n_charges, pb.sectors_A, pb.sectors_B, pb.target)
        dp.create_ops([(o["half"], o["dq"], o["parity"]) for o in pb.ops])
        dp.alloc_resident()
        for i, o in enumerate(pb.ops):
            dp.set_op_host(i, o["blocks"])
        r, c = dp.table[0], dp.table[1]
        bc = np.ones((len(pb.terms), len(r)))
        for (k, blk), v in pb.block_coef.items():
            bc[k, [i for i in range(len(r)) if (int(r[i]), int(c[i])) == blk][0]] = v
        dp.build(pb.terms, block_coef=bc, **opts)
        return dp

    pb = heff.problem_from_workload(medium_spinless())
    rng = np.random.default_rng(5)
    pb.block_coef = {(k, blk): (0.0 if rng.random() < 0.2 else float(rng.normal())) for k in range(len(pb.terms))
                     for blk in pb.psi_blocks() if rng.random() < 0.7}
    for opts in ({}, {"order_policy": 2}):
        dp = on_device(pb, **opts)
        assert rel_max(dp.to_blocks(dp.apply(dp.psi_from_host(pb.psi))), heff.sigma_blockwise(pb)) <= TOL_SIGMA
        assert dp.heff.n_tasks == len(heff.enumerate_tasks(pb))
    dim, H = dimer_singlet_problem()
    dp = on_device(dim)
    x = dp.psi_from_host(dim.psi)
    assert rel_max(dp.to_blocks(dp.apply(x)), heff.sigma_dense(dim)) <= TOL_SIGMA
    dav = dp.davidson(m_max=3, tol=1e-12, max_iter=50)
    dav.start(x)
    theta, rn, n_apply, ok = dav.solve(None)
    E0 = float(golden_table("closed_forms.txt")["hubbard_dimer_E0_U4"])
    assert ok and abs(theta - E0) <= 1e-9


@pytest.mark.parametrize("kernel", [0, 4])
def test_balanced_tiles_at_edge_dims(kernel):
    """Sector sizes on both sides of every tile-count boundary (64/65, 128/129, one row, a 16-multiple, a
    4-multiple that is no 8-multiple …): the balanced tiling (tile origins at multiples of 16, a tile's
    fragments split evenly over the warp rows/columns, internal.h tile_cuts) must cover each block exactly
    once, padding rows and columns included."""
    dims_a = [1, 64, 65, 129, 12, 100, 128, 200, 17]
    dims_b = [130, 16, 1, 63, 192, 66, 20, 127, 72]
    secA = [((q,), d) for q, d in enumerate(dims_a)]
    secB = [((q,), d) for q, d in enumerate(dims_b)]
    wl = wlmod.Workload("edge_dims", 23, 1, secA, secB, (8,))
    for k, dlt in enumerate([0, 1, -1, 2, -2, 3, -3, 1]):
        wl.ops.append(wlmod.OpSpec("A", (dlt,), dlt & 1, False, "one", f"L{k}"))
        wl.ops.append(wlmod.OpSpec("B", (-dlt,), dlt & 1, False, "one", f"R{k}"))
        wl.terms.append(wlmod.TermSpec(2 * k, 2 * k + 1, 0.5 - 0.1 * k, False, False, "syn"))
        wl.terms.append(wlmod.TermSpec(2 * k, 2 * k + 1, 0.25 + 0.1 * k, True, True, "syn^T"))
    pb = heff.problem_from_workload(wl)
    ref = heff.sigma_blockwise(pb)
    for opts in ({}, {"split_waves": 64}, {"order_policy": 2}):
        dp = device_problem(pb, kernel=kernel, **opts)
        sigma = dp.apply(dp.psi_from_host(pb.psi))
        assert rel_max(dp.to_blocks(sigma), ref) <= TOL_SIGMA, opts
        assert padding_is_zero(dp, sigma)
        assert rel_max(dp.to_blocks(dp.diag()), heff.diagonal_blockwise(pb)) <= 1e-13
