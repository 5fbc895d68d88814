"""Pins for oracle/fock.py and oracle/lattice.py (T0): anticommutators, an
independent bit-string construction, closed forms, stored ED energies, spectrum
invariance under mode rotation."""
import math

import numpy as np
import pytest

from oracle import fock, lattice
from _util import golden_table


def test_anticommutation_relations():
    # {c_i, c_j} = 0, {c†_i, c_j} = δ_ij
    n = 5
    c = fock.annihilators(n)
    I = np.eye(2 ** n)
    for i in range(n):
        for j in range(n):
            ci, cj = c[i].toarray(), c[j].toarray()
            assert np.abs(ci @ cj + cj @ ci).max() == 0.0
            assert np.abs(ci.T @ cj + cj @ ci.T - (I if i == j else 0 * I)).max() == 0.0


def test_basis_convention_mode0_most_significant():
    c = fock.annihilators(3)
    vac = np.zeros(8)
    vac[0] = 1.0
    # c†_0 |vac> = |100> = index 4 ; c†_1 c†_2|vac> = |011> = index 3, sign +
    assert (c[0].T @ vac)[4] == 1.0
    assert (c[1].T @ (c[2].T @ vac))[3] == 1.0
    # c†_2 c†_1 |vac> = -|011>
    assert (c[2].T @ (c[1].T @ vac))[3] == -1.0


def test_kronecker_vs_bitstring_hamiltonian():
    rng = np.random.default_rng(11)
    n = 5
    T = rng.normal(size=(n, n))
    V = rng.normal(size=(n, n, n, n))
    H1 = fock.hamiltonian(T, V).toarray()
    H2 = fock.hamiltonian_bits(T, V)
    assert np.abs(H1 - H2).max() < 1e-12
    assert np.abs(H1).max() > 1.0


def test_hermitian_and_number_conserving():
    T, V, mc = lattice.spinless_tV(3)
    H = fock.hamiltonian(T, V).toarray()
    assert np.abs(H - H.T).max() == 0.0
    N = fock.occupations(9).sum(axis=1)
    # [H, N] = 0  <=>  H only connects states of equal N
    r, c = np.nonzero(H)
    assert np.all(N[r] == N[c])


def test_torus_bond_counts():
    nn, nnn = lattice.torus_bonds(4)
    assert len(nn) == 32 and len(nnn) == 32
    assert sorted(lattice.snake_position(1, c, 4) for c in range(4)) == [4, 5, 6, 7]
    assert lattice.snake_position(1, 0, 4) == 7      # odd rows run backwards (r4)


def test_free_fermion_levels_closed_form():
    g = golden_table("closed_forms.txt")
    want = np.array([float(x) for x in g["torus4_levels"].split()])
    T, V, _ = lattice.spinless_tV(4, 1.0, 0.4, 0.0)
    got = np.sort(np.linalg.eigvalsh(T))
    ks = [2 * math.pi * i / 4 for i in range(4)]
    formula = np.sort([-2 * (math.cos(kx) + math.cos(ky)) - 4 * 0.4 * math.cos(kx) * math.cos(ky)
                       for kx in ks for ky in ks])
    assert np.abs(got - formula).max() < 1e-12
    assert np.abs(got - want).max() < 1e-12
    assert abs(got[:8].sum() - float(g["torus4_free_E0_N8"])) < 1e-12


def test_free_fermion_many_body_energy():
    # V = 0: E0(N) = sum of the N lowest one-body levels, through the full Fock-space route
    T, V, mc = lattice.spinless_tV(3, 1.0, 0.4, 0.0)
    lev = np.sort(np.linalg.eigvalsh(T))
    for N in (3, 4, 5):
        assert abs(fock.ground_energy(T, V, mc, (N,)) - lev[:N].sum()) < 1e-11


def test_hubbard_dimer_closed_form():
    g = golden_table("closed_forms.txt")
    T, V, mc = lattice.hubbard_tV(None, 1.0, 4.0, bonds=[(0, 1)], n_sites=2)
    E = fock.ground_energy(T, V, mc, (1, 1))
    assert abs(E - (4 - math.sqrt(16 + 16)) / 2) < 1e-12
    assert abs(E - float(g["hubbard_dimer_E0_U4"])) < 1e-12


def test_hubbard_U0_is_two_free_species():
    T, V, mc = lattice.hubbard_tV(None, 1.0, 0.0, bonds=[(0, 1), (1, 2), (2, 3), (3, 0), (0, 2)], n_sites=4)
    lev = np.sort(np.linalg.eigvalsh(T[0::2, 0::2]))
    assert abs(fock.ground_energy(T, V, mc, (2, 1)) - (lev[:2].sum() + lev[:1].sum())) < 1e-11


def test_hubbard_interaction_counts_double_occupancy():
    # t = 0: H = U Σ n↑n↓ is diagonal with eigenvalue U · (number of doubly occupied sites)
    T, V, mc = lattice.hubbard_tV(None, 0.0, 3.0, bonds=[(0, 1)], n_sites=2)
    H = fock.hamiltonian(T, V).toarray()
    occ = fock.occupations(4)
    dbl = occ[:, 0] * occ[:, 1] + occ[:, 2] * occ[:, 3]
    assert np.abs(H - np.diag(3.0 * dbl)).max() == 0.0


def test_stored_ed_energies_3x3():
    g = golden_table("ed_energies.txt")
    for N in (4, 5):
        T, V, mc = lattice.spinless_tV(3)
        assert abs(fock.ground_energy(T, V, mc, (N,)) - float(g[f"spinless_3x3_N{N}"])) < 1e-10


def test_stored_ed_energy_4x4_bitstring_cross_check():
    """The 12870-dim N=8 sector of the 4×4 torus, built a second way (explicit
    hopping / interaction rules on bit strings, no Jordan-Wigner matrices)."""
    import scipy.sparse as sp
    from scipy.sparse.linalg import eigsh
    g = golden_table("ed_energies.txt")
    L, n, N = 4, 16, 8
    nn, nnn = lattice.torus_bonds(L)
    states = [s for s in range(2 ** n) if bin(s).count("1") == N]
    index = {s: i for i, s in enumerate(states)}
    bit = lambda p: 1 << (n - 1 - p)
    rows, cols, vals = [], [], []
    for s in states:
        diag = 0.0
        for i, j in nn:
            if s & bit(i) and s & bit(j):
                diag += 0.8
        rows.append(index[s]); cols.append(index[s]); vals.append(diag)
        for bonds, amp in ((nn, -1.0), (nnn, -0.4)):
            for i, j in bonds:
                for a, b in ((i, j), (j, i)):        # c†_a c_b
                    if (s & bit(b)) and not (s & bit(a)):
                        lo, hi = min(a, b), max(a, b)
                        between = sum(1 for p in range(lo + 1, hi) if s & bit(p))
                        s2 = (s ^ bit(b)) | bit(a)
                        rows.append(index[s2]); cols.append(index[s]); vals.append(amp * (-1) ** between)
    H = sp.csr_matrix((vals, (rows, cols)), shape=(len(states), len(states)))
    assert abs(H - H.T).max() < 1e-14
    E = np.sort(eigsh(H, k=3, which="SA", tol=1e-12, ncv=48)[0])[0]
    assert abs(E - float(g["spinless_4x4_N8"])) < 1e-9


def test_mode_rotation_leaves_spectrum_intact():
    # "a unitary transformation on the Hamiltonian leaves the energy spectrum intact"
    T, V, mc = lattice.spinless_tV(3)
    U = lattice.rotation_matrix(9, seed=3)
    assert np.abs(U.T @ U - np.eye(9)).max() < 1e-13
    Tr, Vr = lattice.rotate(T, V, U)
    assert np.count_nonzero(np.abs(Vr) > 1e-12) > 1000      # the rotated V is dense
    idx = fock.sector_indices(9, mc, (4,))
    e0 = np.linalg.eigvalsh(fock.restrict(fock.hamiltonian(T, V), idx).toarray())
    e1 = np.linalg.eigvalsh(fock.restrict(fock.hamiltonian(Tr, Vr), idx).toarray())
    assert np.abs(e0 - e1).max() < 1e-10


def test_hubbard_spin_restricted_rotation_spectrum():
    T, V, mc = lattice.hubbard_tV(None, 1.0, 4.0, bonds=[(0, 1), (1, 2), (2, 0)], n_sites=3)
    U2 = lattice.spin_rotation(lattice.rotation_matrix(3, seed=4))
    Tr, Vr = lattice.rotate(T, V, U2)
    idx = fock.sector_indices(6, mc, (2, 1))
    e0 = np.linalg.eigvalsh(fock.restrict(fock.hamiltonian(T, V), idx).toarray())
    e1 = np.linalg.eigvalsh(fock.restrict(fock.hamiltonian(Tr, Vr), idx).toarray())
    assert np.abs(e0 - e1).max() < 1e-10


@pytest.mark.parametrize("n,mc,target", [(8, [(1,)] * 8, (4,)), (8, [(1, 0), (0, 1)] * 4, (2, 2)), (9, [(1,)] * 9, (5,)),
                                         (7, [(1, 0), (0, 1)] * 3 + [(1, 0)], (2, 1))])
def test_sector_hamiltonian_equals_restricted_kronecker_hamiltonian(n, mc, target):
    """fock.hamiltonian_sector (bit-string actions inside one charge sector) against the Kronecker construction
    restricted to the same states, on fully random NON-symmetric t and V (every index order matters, every sign)."""
    rng = np.random.default_rng(n)
    T, V = rng.normal(size=(n, n)), rng.normal(size=(n,) * 4)
    rows, H = fock.hamiltonian_sector(T, V, np.array(mc), target)
    ref = fock.restrict(fock.hamiltonian(T, V), fock.sector_indices(n, np.array(mc), target))
    assert np.array_equal(rows, fock.sector_indices(n, np.array(mc), target))
    assert abs(H - ref).max() <= 1e-13 * abs(ref).max() and abs(ref).max() > 1.0


def test_sector_action_matches_single_state_action():
    """The vectorised string action against apply_string_bits state by state (signs and target states)."""
    n = 6
    cols = np.arange(2 ** n)
    occ = fock.occupations(n)
    for string in ([("-", 2)], [("+", 4)], [("-", 1), ("-", 3)], [("+", 0), ("+", 5), ("-", 2), ("-", 4)]):
        M = fock.sector_action(string, n, cols).toarray()
        for c in cols:
            s, new = fock.apply_string_bits(string, tuple(occ[c]))
            col = np.zeros(2 ** n)
            if s:
                col[int("".join(map(str, new)), 2)] = s
            assert np.array_equal(M[:, c], col)


@pytest.mark.slow
def test_rotated_4x4_sector_hamiltonian_keeps_the_ed_energy():
    """The mode-rotated 4×4 torus (dense t, V: the workload of the K = 154 twin) built inside the N = 8 sector
    is symmetric and has the exact-diagonalisation ground energy of the real-space model (the
    rotation is a unitary transformation of the modes, tests/golden/ed_energies.txt spinless_4x4_N8)."""
    from scipy.sparse.linalg import eigsh
    T, V, mc = lattice.spinless_tV(4)
    Tr, Vr = lattice.rotate(T, V, lattice.rotation_matrix(16, seed=7))
    rows, H = fock.hamiltonian_sector(Tr, Vr, mc, (8,))
    assert H.shape == (12870, 12870) and abs(H - H.T).max() <= 1e-12
    e0 = np.sort(eigsh(H, k=2, which="SA", tol=1e-12)[0])[0]
    assert abs(e0 - (-8.378565104009)) <= 1e-9
