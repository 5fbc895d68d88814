"""-m gpu parity of dmrgk_heff_expect: per-pair expectation values
⟨ψ, c_k (L_k ⊗ R_k) ψ⟩ from the grouped GEMM kernel + fused dots against oracle.heff.expectation_per_pair,
and the one-particle reduced density matrix of a DMRG bond against its Fock-space definition."""
import numpy as np
import pytest

import workloads as wlmod
from oracle import dmrg, heff
from test_oracle_enlarge import spinless_3x3, hubbard_ring
from _rdm import rdm_pairs, rdm_fock
from _gpu import device_problem

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.mark.parametrize("opts", [{}, {"t_chunk_bytes": 1 << 20}, {"order_policy": 2}])
def test_per_pair_expectations_vs_oracle(opts):
    thin = lambda fam, i: fam in ("F1", "F2") or i % 5 == 0
    wl = wlmod.lattice_workload("spinless", 10, 600, seed=13, width2=4.0, keep=thin)
    pb = heff.problem_from_workload(wl)
    ref = heff.expectation_per_pair(pb)
    dp = device_problem(pb, per_pair_output=1, **opts)
    psi = dp.psi_from_host(pb.psi)
    got = dp.expect(psi, len(pb.terms)).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max()
    again = dp.expect(psi, len(pb.terms)).cpu().numpy()
    assert np.array_equal(got, again)                          # fixed-order dots: bit-reproducible
    if "t_chunk_bytes" in opts:
        assert dp.heff.n_chunks > 1
    # a per-pair plan is not an H_eff plan
    from paper_2311_14106_b200 import dmrgk
    with pytest.raises(dmrgk.DmrgkError) as e:
        dp.apply(psi)
    assert e.value.status == dmrgk.ESTATE
    # and the K numbers add up to ⟨ψ, H_eff ψ⟩ of the summed plan
    full = device_problem(pb)
    x = full.psi_from_host(pb.psi)
    assert abs(float(torch.dot(x, full.apply(x))) - got.sum()) <= 1e-10 * np.abs(got).sum()


@pytest.mark.parametrize("make,bond,N", [(spinless_3x3(64), 4, 4), (hubbard_ring(8), 1, 4)])
def test_one_particle_rdm_of_a_dmrg_bond(make, bond, N):
    T, V, mc, site_modes, target, D = make
    d = dmrg.SimpleDMRG(T, V, mc, site_modes, target, D=D, seed=2)
    d.warmup_to(bond)
    space = d.space_at(bond)
    Heff, P = d.heff_at(space)
    E, x = dmrg.lowest_eigenpair(Heff)
    pb, labels = rdm_pairs(d, space)
    pb.psi = dmrg.vec_to_blocks(space, x)
    dp = device_problem(pb, per_pair_output=1)
    got = dp.expect(dp.psi_from_host(pb.psi), len(pb.terms)).cpu().numpy()
    gamma = rdm_fock(d, space, x)
    listed = set(labels)
    assert all(abs(gamma[i, j]) <= 1e-12 for i in range(d.n) for j in range(i, d.n) if (i, j) not in listed)
    for (i, j), v in zip(labels, got):
        assert abs(v - gamma[i, j]) <= 1e-11, (i, j)
    assert abs(sum(v for (i, j), v in zip(labels, got) if i == j) - N) <= 1e-11


@pytest.mark.parametrize("make,bond,N", [(spinless_3x3(64), 4, 4), (spinless_3x3(6), 3, 4), (hubbard_ring(8), 1, 4)])
def test_two_particle_rdm_of_a_dmrg_bond(make, bond, N):
    """Γ_ijkl = ⟨c†_i c†_j c_k c_l⟩, i < j, k < l (the two-mode quantities of PAPER.md:88), through
    dmrgk_heff_expect on the pair list of the strings split across the cut — one pair per charge-conserving
    string, reordering sign as the coefficient — against the Fock-space definition at 1e-11, plus the partial
    trace Σ_j Γ_ijjk = (N − 1) γ_ik against the Fock-space one-particle matrix."""
    from _rdm import rdm2_strings, rdm2_fock, string_pairs
    T, V, mc, site_modes, target, D = make
    d = dmrg.SimpleDMRG(T, V, mc, site_modes, target, D=D, seed=2)
    d.warmup_to(bond)
    space = d.space_at(bond)
    Heff, P = d.heff_at(space)
    E, x = dmrg.lowest_eigenpair(Heff)
    labels, strings = rdm2_strings(d.n)
    pb, kept = string_pairs(d, space, strings)
    pb.psi = dmrg.vec_to_blocks(space, x)
    dp = device_problem(pb, per_pair_output=1)
    got = dp.expect(dp.psi_from_host(pb.psi), len(pb.terms)).cpu().numpy()
    ref = rdm2_fock(d, space, x, labels)
    assert np.abs(got - ref[kept]).max() <= 1e-11
    assert np.abs(got - heff.expectation_per_pair(pb)).max() <= 1e-11
    n = d.n
    G = np.zeros((n, n, n, n))
    for idx, v in zip(kept, got):
        i, j, k, l = labels[idx]
        G[i, j, k, l], G[j, i, k, l], G[i, j, l, k], G[j, i, l, k] = v, -v, -v, v
    assert np.abs(np.einsum("ijjk->ik", G) - (N - 1) * rdm_fock(d, space, x)).max() <= 1e-10
