"""-m gpu parity of the SU(2) spin-adapted H_eff for a singlet target.

The oracle (oracle/su2.py) hands over what a spin-adapted DMRG would: sector lists in multiplets, the reduced
matrix elements of the tensor-operator pairs, the pair list with each pair's rank.  The recoupling scalars are
the LIBRARY side's (paper_2311_14106_b200/su2.py, closed form) — the oracle's brute-force table is not passed
in.  σ is compared with the oracle's blockwise tier and with the definition Cᵀ H C ψ at 1e-11, the Davidson
energy with the lowest singlet level of the Fock-space Hamiltonian at 1e-9."""
import numpy as np
import pytest

from oracle import su2 as osu2, heff, fock
from _gpu import rel_max, padding_is_zero, TOL_SIGMA, TOL_ENERGY
from test_oracle_su2 import hubbard, singlet_spectrum_from_S2

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.mark.parametrize("R,Cn,nA,rotated,keep", [(2, 2, 2, True, None), (2, 3, 3, False, None), (2, 3, 3, True, None),
                                                   (2, 3, 2, True, None), (2, 3, 3, True, 0.6)])
def test_singlet_heff_sigma_and_energy(R, Cn, nA, rotated, keep):
    from paper_2311_14106_b200 import su2
    T, V, mc = hubbard(R, Cn, rotated)
    n = R * Cn
    pb, multA, multB, groups, defects = osu2.reduced_problem(T, V, nA, n, keep=keep, seed=5)
    rng = np.random.default_rng(8)
    pb.psi = {(a, b): rng.normal(size=(pb.sectors_A[a][1], pb.sectors_B[b][1])) for (a, b) in pb.psi_blocks()}
    pairs = [(L, Rr, c, k2) for (L, Rr, c, _, _), k2 in zip(pb.terms, pb.ranks)]
    for opts in ({}, {"order_policy": 2}):
        dp = su2.singlet_problem(pb.sectors_A, pb.sectors_B, n, pb.ops, pairs, **opts)
        sigma = dp.apply(dp.psi_from_host(pb.psi))
        got = dp.to_blocks(sigma)
        assert rel_max(got, heff.sigma_blockwise(pb)) <= TOL_SIGMA            # the method, step by step
        C = osu2.singlet_isometry(multA, multB, n)
        H_def = C.T @ (fock.hamiltonian(T, V) @ C)                             # the definition
        ref = heff.vec_to_psi(pb, H_def @ heff.psi_to_vec(pb))
        assert rel_max(got, ref) <= TOL_SIGMA
        assert padding_is_zero(dp, sigma)
        assert rel_max(dp.to_blocks(dp.diag()), heff.vec_to_psi(pb, np.diag(H_def).copy())) <= 1e-12
    # spin-adapted dimension: multiplets, fewer than the U(1) states of the same half
    assert sum(d for _, d in pb.sectors_A) < 4 ** nA
    dav = dp.davidson(m_max=16, tol=1e-9, max_iter=3000)
    dav.start(dp.psi_from_host(pb.psi))
    theta, rn, n_apply, ok = dav.solve(None)
    assert ok
    E = np.linalg.eigvalsh(H_def)[0]
    assert abs(theta - E) <= TOL_ENERGY * max(1.0, abs(E))
    E_singlet = singlet_spectrum_from_S2(T, V, n, n)[0]
    if keep is None:
        assert abs(theta - E_singlet) <= TOL_ENERGY * max(1.0, abs(E_singlet))
    else:
        assert theta >= E_singlet - 1e-9                                        # variational


def oracle_block_coef(wl, pb):
    """The oracle's recoupling table of a spin-adapted workload: brute-force Clebsch–Gordan sums
    (oracle.su2.recoupling_singlet) times the Jordan–Wigner sign, per (pair, input ψ block)."""
    table = {}
    for k, ((L, R, c, tL, tR), k2) in enumerate(zip(pb.terms, wl.ranks)):
        for (a, b) in pb.psi_blocks():
            N, tS = pb.sectors_A[a][0]
            if L is None or R is None:
                table[(k, (a, b))] = 1.0
                continue
            d2 = pb.ops[L]["dq"][1] * (-1 if tL else 1)
            x = osu2.recoupling_singlet(tS, tS + d2, k2) if tS + d2 >= 0 else 0.0
            table[(k, (a, b))] = (-x if (pb.ops[L]["parity"] and N % 2) else x)
    return table


@pytest.mark.parametrize("opts", [{}, {"split_waves": 64}, {"order_policy": 2}, {"kernel": 5}])
def test_su2_structured_workload_vs_oracle(opts):
    """The spin-adapted workload of `bench.py --op su2`, scaled down (6 orbitals per half, 900 multiplets, synthetic
    reduced matrix elements, sectors up to 2S = 6, all families, h.c. partners through the transpose flags): σ with the
    library's closed-form recoupling table against the oracle's blockwise tier with the brute-force table."""
    import workloads as wlmod
    from paper_2311_14106_b200 import problem, su2
    thin = lambda fam, i: fam in ("F1", "F2") or i % 3 == 0
    wl = wlmod.su2_singlet_workload(6, 900, seed=16, keep=thin)
    pb = heff.problem_from_workload(wl)
    pb.block_coef = oracle_block_coef(wl, pb)
    assert any(v == 0.0 for v in pb.block_coef.values())            # triangle rule: S = 0 → S′ = 0 through a rank-1 pair
    ref = heff.sigma_blockwise(pb)
    terms = [(t.L, t.R, t.coef, t.trans_L, t.trans_R) for t in wl.terms]
    psi_a = [a for (a, _, _, _, _) in wlmod.psi_block_table(wl.sectors_A, wl.sectors_B, wl.target)]
    table = su2.block_coef_table(wl.sectors_A, psi_a, su2.pair_meta(wl.ops, terms, wl.ranks))
    dp = problem.from_workload(wl, block_coef=table, **opts)
    psi = dp.psi_fill(wl.seed, wlmod.PSI_STREAM)
    sigma = dp.apply(psi)
    assert rel_max(dp.to_blocks(sigma), ref) <= TOL_SIGMA
    assert padding_is_zero(dp, sigma)
    assert dp.heff.n_tasks == len(heff.enumerate_tasks(pb))
    assert dp.heff.flops_alg == heff.flops_alg(pb)


def test_su2_workload_of_the_bench_sampled_blocks():
    """`bench.py --op su2` at its full size (190 sectors (N, 2S), 12288 multiplets, K = 2702 pairs, 99 GB of
    reduced operators), in the launch configuration that op times: σ on ≥ 8 sampled output blocks — the largest,
    the smallest, both edges of the sector range — against the oracle's blockwise tier on operator blocks read
    back D2H, the oracle's recoupling scalars by brute-force Clebsch–Gordan sums, the library's in closed form.
    Error against the oracle's scale (1e-11) and per block (1e-10)."""
    import workloads as wlmod
    from paper_2311_14106_b200 import problem, su2
    from _gpu import DeviceInputs, sample_output_blocks, oracle_sigma_on_block, TOL_BLOCK
    wl = wlmod.su2_singlet_workload()
    terms = [(t.L, t.R, t.coef, t.trans_L, t.trans_R) for t in wl.terms]
    psi_a = [a for (a, _, _, _, _) in wlmod.psi_block_table(wl.sectors_A, wl.sectors_B, wl.target)]
    table = su2.block_coef_table(wl.sectors_A, psi_a, su2.pair_meta(wl.ops, terms, wl.ranks))
    dp = problem.from_workload(wl, block_coef=table)
    inputs = DeviceInputs(wl, dp)
    picks = sample_output_blocks(dp.table)
    assert len(picks) >= 8
    psi = dp.psi_fill(wl.seed, wlmod.PSI_STREAM)
    psi_blocks = dp.to_blocks(psi)
    got = dp.to_blocks(dp.apply(psi))

    def coef_of(k, blk):
        L, R, _, tL, _ = terms[k]
        if L is None or R is None:
            return 1.0
        N, tS = wl.sectors_A[blk[0]][0]
        d2 = wl.ops[L].dq[1] * (-1 if tL else 1)
        x = osu2.recoupling_singlet(tS, tS + d2, wl.ranks[k]) if tS + d2 >= 0 else 0.0
        return -x if (wl.ops[L].parity and N % 2) else x

    refs = {k: oracle_sigma_on_block(wl, inputs, k[0], k[1], psi_blocks, coef_of=coef_of) for k in picks}
    scale = max(np.abs(v).max() for v in refs.values())
    for k, ref in refs.items():
        err = np.abs(got[k] - ref).max()
        assert err <= TOL_SIGMA * scale, (k, err / scale)
        assert err <= TOL_BLOCK * np.abs(ref).max(), (k, "per-block")
    assert inputs.checked > 0
