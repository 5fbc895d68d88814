"""Pin of oracle.heff.expectation_per_pair: with the pair list of c†_i c_j at a DMRG bond it gives the
one-particle reduced density matrix of the state, γ_ij = ⟨Ψ|c†_i c_j|Ψ⟩ built in Fock space (PAPER.md:88,
166); Tr γ = N; and the per-pair values add up to ⟨ψ, H_eff ψ⟩ of the whole list."""
import numpy as np
import pytest

from oracle import dmrg, heff
from test_oracle_enlarge import spinless_3x3, hubbard_ring
from _rdm import rdm_pairs, rdm_fock


@pytest.mark.parametrize("make,bond,N", [(spinless_3x3(64), 4, 4), (spinless_3x3(6), 3, 4), (hubbard_ring(8), 1, 4)])
def test_one_particle_rdm_from_pair_expectations(make, bond, N):
    T, V, mc, site_modes, target, D = make
    d = dmrg.SimpleDMRG(T, V, mc, site_modes, target, D=D, seed=2)
    d.warmup_to(bond)
    space = d.space_at(bond)
    Heff, P = d.heff_at(space)
    E, x = dmrg.lowest_eigenpair(Heff)
    pb, labels = rdm_pairs(d, space)
    pb.psi = dmrg.vec_to_blocks(space, x)
    e = heff.expectation_per_pair(pb)
    gamma = rdm_fock(d, space, x)
    listed = set(labels)
    assert all(abs(gamma[i, j]) <= 1e-12 for i in range(d.n) for j in range(i, d.n) if (i, j) not in listed)
    for (i, j), v in zip(labels, e):
        assert abs(v - gamma[i, j]) <= 1e-12, (i, j)
    assert abs(sum(v for (i, j), v in zip(labels, e) if i == j) - N) <= 1e-12
    # additivity: Σ_k e_k = ⟨ψ, (Σ_k pairs) ψ⟩
    sig = heff.sigma_blockwise(pb)
    assert abs(sum(e) - sum(float(np.sum(sig[k] * pb.psi[k])) for k in pb.psi)) <= 1e-11


def _bond_state(make, bond):
    T, V, mc, site_modes, target, D = make
    d = dmrg.SimpleDMRG(T, V, mc, site_modes, target, D=D, seed=2)
    d.warmup_to(bond)
    space = d.space_at(bond)
    Heff, P = d.heff_at(space)
    E, x = dmrg.lowest_eigenpair(Heff)
    return d, space, x


def test_split_string_signs_by_hand():
    """A|B = modes {0,1}|{2,3}.  c†_0 c†_2 c_1 c_3: c_1 passes one B-operator → −; c†_2 c†_3 c_0 c_1: each of the
    two A-operators passes two → +; c†_2 c†_0 c_3 c_1: c†_0 passes one, c_1 passes two → −."""
    from _rdm import split_string
    s = lambda *modes: [(m, dg) for m, dg in zip(modes, (True, True, False, False))]
    assert split_string(s(0, 2, 1, 3), 2) == (-1.0, [(0, True), (1, False)], [(0, True), (1, False)])
    assert split_string(s(2, 3, 0, 1), 2) == (1.0, [(0, False), (1, False)], [(0, True), (1, True)])
    assert split_string(s(2, 0, 3, 1), 2)[0] == -1.0
    assert split_string(s(0, 1, 0, 1), 2) == (1.0, s(0, 1, 0, 1), [])


@pytest.mark.parametrize("make,bond,N", [(spinless_3x3(64), 4, 4), (spinless_3x3(6), 3, 4), (hubbard_ring(8), 1, 4)])
def test_two_particle_rdm_from_pair_expectations(make, bond, N):
    """Γ_ijkl = ⟨c†_i c†_j c_k c_l⟩ (i < j, k < l) from oracle.heff.expectation_per_pair on the pair list of the
    strings split across the cut (all of (4|0), (3|1), (2|2), (1|3), (0|4) occur) against the Fock-space
    definition; the partial trace Σ_j Γ_ijjk = (N − 1) γ_ik ties it to the one-particle matrix, Σ_{i<j} Γ_ijij =
    −N(N−1)/2; without the reordering sign it is wrong (control)."""
    from _rdm import rdm2_strings, rdm2_fock, string_pairs
    d, space, x = _bond_state(make, bond)
    labels, strings = rdm2_strings(d.n)
    pb, kept = string_pairs(d, space, strings)
    n_A = space.A.n_modes
    assert {sum(m < n_A for m in lab) for lab in labels} == {0, 1, 2, 3, 4}
    pb.psi = dmrg.vec_to_blocks(space, x)
    e = heff.expectation_per_pair(pb)
    ref = rdm2_fock(d, space, x, labels)
    dropped = sorted(set(range(len(labels))) - set(kept))
    assert np.abs(ref[dropped]).max(initial=0.0) <= 1e-12            # charge-violating strings vanish by symmetry
    assert np.abs(e - ref[kept]).max() <= 1e-12
    assert np.abs(ref).max() > 1e-2
    # full tensor by antisymmetry, then the contractions
    n = d.n
    G = np.zeros((n, n, n, n))
    for idx, v in zip(kept, e):
        i, j, k, l = labels[idx]
        G[i, j, k, l], G[j, i, k, l], G[i, j, l, k], G[j, i, l, k] = v, -v, -v, v
    gamma = rdm_fock(d, space, x)
    assert np.abs(np.einsum("ijjk->ik", G) - (N - 1) * gamma).max() <= 1e-11
    assert abs(sum(G[i, j, i, j] for i in range(n) for j in range(i + 1, n)) + N * (N - 1) / 2) <= 1e-11
    # control: the same list with every reordering sign set to +1 does not give Γ
    plain = heff.Problem(pb.n_charges, pb.sectors_A, pb.sectors_B, pb.target, pb.ops,
                         [(L, R, 1.0, tL, tR) for (L, R, c, tL, tR) in pb.terms], pb.psi)
    assert np.abs(heff.expectation_per_pair(plain) - ref[kept]).max() > 1e-3
