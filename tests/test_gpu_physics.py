"""-m gpu parity on REAL physics beyond config 1's real-space list (SURVEY §8(d) configs 1 and 4,
"scaled-down physics twin"): exported DMRG bonds of mode-rotated lattices, so families F2, F3 and the
off-diagonal F4 pairs reach the device with the values the regrouping of Eq. (1) gives
them, not synthetic ones.  σ at 1e-11 against the definition P†HP ψ (T1) and against the dense
Kronecker form of the exported blocks (T2); Davidson θ at 1e-9 against `eigh` of P†HP.

The twins: the 3×3 spinless torus (t-t′-V, 9 modes, rotated, all of F0-F4 dense) and a 2×3 Hubbard
torus (12 spin-orbitals, two charges (n↑, n↓), same spatial rotation for both spins).
The rotated 4×4 variant (K = 154) of §8(d) — config 1's own bond with the dense term list — runs through
`fock.hamiltonian_sector`, the Hamiltonian built inside the N = 8 sector (the 2^16-dimensional Kronecker
builder would need 16⁴ sparse products).
"""
import numpy as np
import pytest

from oracle import heff, lattice, dmrg, export, fock
from _gpu import device_problem, rel_max, padding_is_zero, TOL_SIGMA, TOL_ENERGY

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def torus_bonds_rect(R, Cn):
    """Nearest-neighbour bonds of an R×Cn torus in snake order (reading r3: per site → right and
    down neighbours, indices mod the extent, no de-duplication)."""
    pos = lambda r, c: r * Cn + (c if r % 2 == 0 else Cn - 1 - c)
    out = []
    for r in range(R):
        for c in range(Cn):
            out.append((pos(r, c), pos(r, (c + 1) % Cn)))
            out.append((pos(r, c), pos((r + 1) % R, c)))
    return out


def spinless_3x3_rotated(D):
    T, V, mc = lattice.spinless_tV(3)
    T, V = lattice.rotate(T, V, lattice.rotation_matrix(9, seed=3))
    d = dmrg.SimpleDMRG(T, V, mc, [[i] for i in range(9)], (4,), D=D, seed=2)
    d.warmup_to(4)
    return d, d.space_at(4), (T, V, mc, (4,))


def hubbard_2x3_rotated(D):
    T, V, mc = lattice.hubbard_tV(None, 1.0, 4.0, bonds=torus_bonds_rect(2, 3), n_sites=6)
    T, V = lattice.rotate(T, V, lattice.spin_rotation(lattice.rotation_matrix(6, seed=4)))
    d = dmrg.SimpleDMRG(T, V, mc, [[2 * i, 2 * i + 1] for i in range(6)], (3, 3), D=D, seed=4)
    d.warmup_to(2)
    return d, d.space_at(2), (T, V, mc, (3, 3))


@pytest.mark.parametrize("make,D,families", [
    (spinless_3x3_rotated, 64, 2 + 2 * 4 + 2 * 5 + 5 * 4 + 25),     # n_A = 5, n_B = 4; untruncated: DMRG exact
    (spinless_3x3_rotated, 6, 2 + 2 * 4 + 2 * 5 + 5 * 4 + 25),      # truncated bases
    (hubbard_2x3_rotated, 16, None),
])
def test_rotated_twin_sigma_and_energy(make, D, families):
    d, space, (T, V, mc, target) = make(D)
    Heff, P = d.heff_at(space)
    x = d.guess_at(space, P)
    pb = export.export_bond(d, space)
    pb.psi = dmrg.vec_to_blocks(space, x)
    if families is not None:
        assert len(pb.terms) == families          # dense basis: no pair is pruned (SURVEY §8.0 K formula)
    assert any(t[3] for t in pb.terms)            # h.c. partners go through the transpose flags
    dp = device_problem(pb)
    sigma = dp.apply(dp.psi_from_host(pb.psi))
    got = dp.to_blocks(sigma)
    # T1: the definition
    ref1 = dmrg.vec_to_blocks(space, Heff @ x)
    assert rel_max(got, ref1) <= TOL_SIGMA
    # T2: dense Kronecker assembly of the same exported blocks
    assert rel_max(got, heff.sigma_dense(pb)) <= TOL_SIGMA
    assert padding_is_zero(dp, sigma)
    # Davidson ground energy against eigh of P†HP, and — when the bases are not truncated — against
    # exact diagonalisation of the Fock-space Hamiltonian in the target sector
    E = np.linalg.eigvalsh(Heff)[0]
    dav = dp.davidson(m_max=16, tol=1e-9, max_iter=3000)
    dav.start(dp.psi_from_host(pb.psi))
    theta, rn, n_apply, ok = dav.solve(None)
    assert ok
    assert abs(theta - E) <= TOL_ENERGY * max(1.0, abs(E))
    E_ed = fock.ground_energy(T, V, mc, target)
    assert theta >= E_ed - 1e-9                    # variational
    if make is spinless_3x3_rotated and D == 64:
        assert abs(theta - E_ed) <= TOL_ENERGY * max(1.0, abs(E_ed))


def test_config1_rotated_twin_K154():
    """SURVEY §8(d) row 1, second workload: the 4×4 spinless torus of config 1 in a mode-rotated basis, where
    t and V are dense and the complementary-operator list of the middle bond has the full K = 154 pairs of the
    formula (2 + 2·8 + 2·8 + 8·7 + 64).  The bases of bond 8|9 are those of config 1's own warm-up sweep
    (any isometry defines a valid P†HP); H is Eq. (1) with the rotated t, V inside the N = 8 sector.
    σ at 1e-11 against the definition P†HPψ (T1) and the per-task oracle (T3); Davidson θ at 1e-9 against eigh
    of P†HP, and not below the exact ground energy of the torus (rotation leaves the spectrum unchanged)."""
    T, V, mc = lattice.spinless_tV(4)
    d = dmrg.SimpleDMRG(T, V, mc, [[i] for i in range(16)], (8,), D=64, seed=1)
    d.warmup_to(7)
    Tr, Vr = lattice.rotate(T, V, lattice.rotation_matrix(16, seed=7))
    rows, H = fock.hamiltonian_sector(Tr, Vr, mc, (8,))
    assert np.array_equal(rows, d.rows)
    d.T, d.V, d.H = Tr, Vr, H
    space = d.space_at(7)
    Heff, P = d.heff_at(space)
    x = d.guess_at(space, P)
    pb = export.export_bond(d, space)
    pb.psi = dmrg.vec_to_blocks(space, x)
    assert len(pb.terms) == 2 + 2 * 8 + 2 * 8 + 8 * 7 + 64 == 154
    assert sum(dim for _, dim in space.sectors_A) == 128
    dp = device_problem(pb)
    sigma = dp.apply(dp.psi_from_host(pb.psi))
    got = dp.to_blocks(sigma)
    assert rel_max(got, dmrg.vec_to_blocks(space, Heff @ x)) <= TOL_SIGMA
    assert rel_max(got, heff.sigma_blockwise(pb)) <= TOL_SIGMA
    assert padding_is_zero(dp, sigma)
    E = np.linalg.eigvalsh(Heff)[0]
    dav = dp.davidson(m_max=16, tol=1e-9, max_iter=3000)
    dav.start(dp.psi_from_host(pb.psi))
    theta, rn, n_apply, ok = dav.solve(None)
    assert ok and abs(theta - E) <= TOL_ENERGY * max(1.0, abs(E))
    assert theta >= -8.378565104009 - 1e-9          # tests/golden/ed_energies.txt spinless_4x4_N8; variational
