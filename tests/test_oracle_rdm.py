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
