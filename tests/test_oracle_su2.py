"""Pins of oracle/su2.py: every step of the spin-adapted method
against something other than itself — Clebsch–Gordan coefficients against angular-momentum matrices and
textbook values, multiplets against S² and S^z, the tensor operators against their commutation relations
(with an SU(2)-breaking control), the Wigner–Eckart reduction by its consistency over all M, and the
assembled reduced H_eff against the DEFINITION Cᵀ H C and against the singlet spectrum obtained from the
null space of S² alone."""
import numpy as np
import pytest
import scipy.linalg

from oracle import su2, fock, lattice, terms as oterms, heff

pytestmark = pytest.mark.filterwarnings("ignore")


def spin_matrices(j2):
    """(J^z, J⁺, J⁻) of spin j = j2/2 in the basis m = j, j−1, …, −j."""
    m = np.arange(j2, -j2 - 1, -2) / 2.0
    j = j2 / 2.0
    Jz = np.diag(m)
    Jp = np.zeros((j2 + 1, j2 + 1))
    for i in range(1, j2 + 1):
        Jp[i - 1, i] = np.sqrt(j * (j + 1) - m[i] * (m[i] + 1))
    return Jz, Jp, Jp.T


@pytest.mark.parametrize("j1,j2", [(1, 1), (2, 1), (2, 2), (3, 2), (4, 3), (1, 0)])
def test_cg_against_angular_momentum_matrices(j1, j2):
    z1, p1, m1 = spin_matrices(j1)
    z2, p2, m2 = spin_matrices(j2)
    I1, I2 = np.eye(j1 + 1), np.eye(j2 + 1)
    Jz = np.kron(z1, I2) + np.kron(I1, z2)
    Jp = np.kron(p1, I2) + np.kron(I1, p2)
    Jm = Jp.T
    J2 = Jz @ Jz + 0.5 * (Jp @ Jm + Jm @ Jp)
    vec = lambda J, M: np.array([[su2.cg(j1, a, j2, b, J, M) for b in range(j2, -j2 - 1, -2)] for a in range(j1, -j1 - 1, -2)]).ravel()
    total = 0
    for J in range(abs(j1 - j2), j1 + j2 + 1, 2):
        for M in range(J, -J - 1, -2):
            v = vec(J, M)
            assert abs(v @ v - 1.0) < 1e-13
            assert np.abs(J2 @ v - (J / 2) * (J / 2 + 1) * v).max() < 1e-12
            assert np.abs(Jz @ v - (M / 2) * v).max() < 1e-12
            if M > -J:      # Condon–Shortley: J⁻|J M⟩ = +√(J(J+1) − M(M−1)) |J M−1⟩
                c = np.sqrt((J / 2) * (J / 2 + 1) - (M / 2) * (M / 2 - 1))
                assert np.abs(Jm @ v - c * vec(J, M - 2)).max() < 1e-12
            total += 1
        assert su2.cg(j1, j1, j2, J - j1, J, J) > 0          # ⟨j1 j1 j2 (J − j1)|J J⟩ > 0
    assert total == (j1 + 1) * (j2 + 1)


def test_cg_textbook_values():
    r = np.sqrt
    assert abs(su2.cg(1, 1, 1, -1, 0, 0) - 1 / r(2)) < 1e-15          # ⟨½ ½ ½ −½|0 0⟩
    assert abs(su2.cg(1, -1, 1, 1, 0, 0) + 1 / r(2)) < 1e-15
    assert abs(su2.cg(1, 1, 1, -1, 2, 0) - 1 / r(2)) < 1e-15
    assert abs(su2.cg(2, 0, 2, 0, 4, 0) - r(2 / 3)) < 1e-15           # ⟨1 0 1 0|2 0⟩
    assert abs(su2.cg(2, 2, 2, -2, 0, 0) - 1 / r(3)) < 1e-15          # ⟨1 1 1 −1|0 0⟩
    assert abs(su2.cg(2, 0, 2, 0, 2, 0)) < 1e-15                      # ⟨1 0 1 0|1 0⟩ = 0
    assert abs(su2.cg(2, 2, 1, -1, 1, 1) - r(2 / 3)) < 1e-15          # ⟨1 1 ½ −½|½ ½⟩
    assert su2.cg(2, 2, 2, 2, 2, 4) == 0.0 and su2.cg(1, 1, 1, 1, 0, 2) == 0.0


@pytest.mark.parametrize("n_sites", [1, 2, 3])
def test_multiplets_are_orthonormal_eigenstates_of_S2_Sz_N(n_sites):
    mult = su2.multiplets(n_sites)
    Sp, Sm, Sz, Nop = su2.spin_operators(n_sites)
    S2 = (Sz @ Sz + 0.5 * (Sp @ Sm + Sm @ Sp)).toarray()
    cols, count = [], 0
    for (N, tS), V in mult.items():
        for a in range(V.shape[1]):
            for i in range(tS + 1):
                v = V[:, a, i]
                M = (tS - 2 * i) / 2
                assert np.abs(S2 @ v - (tS / 2) * (tS / 2 + 1) * v).max() < 1e-12
                assert np.abs(Sz @ v - M * v).max() < 1e-12
                assert np.abs(Nop @ v - N * v).max() < 1e-12
                if i < tS:
                    c = np.sqrt((tS / 2) * (tS / 2 + 1) - M * (M - 1))
                    assert np.abs(Sm @ v - c * V[:, a, i + 1]).max() < 1e-12
                cols.append(v)
                count += 1
    assert count == 4 ** n_sites                                    # the multiplets exhaust the Fock space
    Q = np.array(cols)
    assert np.abs(Q @ Q.T - np.eye(count)).max() < 1e-12
    if n_sites == 1:                                                 # |0⟩, the doublet, |↑↓⟩ (D = 3 where U(1) has 4)
        assert {k: v.shape[1] for k, v in mult.items()} == {(0, 0): 1, (1, 1): 1, (2, 0): 1}


def torus_bonds_rect(R, Cn):
    pos = lambda r, c: r * Cn + (c if r % 2 == 0 else Cn - 1 - c)
    out = []
    for r in range(R):
        for c in range(Cn):
            out.append((pos(r, c), pos(r, (c + 1) % Cn)))
            out.append((pos(r, c), pos((r + 1) % R, c)))
    return out


def hubbard(R, Cn, rotated, U=4.0):
    n = R * Cn
    T, V, mc = lattice.hubbard_tV(None, 1.0, U, bonds=torus_bonds_rect(R, Cn), n_sites=n)
    if rotated:      # the same spatial rotation for both spins keeps SU(2) and makes t, V dense
        T, V = lattice.rotate(T, V, lattice.spin_rotation(lattice.rotation_matrix(n, seed=4)))
    return T, V, mc


@pytest.mark.parametrize("R,Cn,nA,rotated", [(2, 2, 2, False), (2, 2, 2, True), (2, 2, 1, True), (1, 3, 1, True)])
def test_tensor_pairs_reassemble_H_and_are_standard_tensors(R, Cn, nA, rotated):
    T, V, mc = hubbard(R, Cn, rotated)
    n = R * Cn
    groups = su2.tensor_groups(T, V, nA)
    H = fock.hamiltonian(T, V)
    assert abs(su2.assemble_groups(groups, nA, n - nA) - H).max() < 1e-12
    for g in groups:
        if g.ident:
            continue
        assert su2.tensor_defect(g.T, g.k2, nA) < 1e-12, (g.family, g.label, "A")
        assert su2.tensor_defect(g.U(), g.k2, n - nA) < 1e-12, (g.family, g.label, "B")
    assert {g.k2 for g in groups} == {0, 1, 2}


def test_tensor_defect_detects_broken_spin_symmetry_and_wrong_phases():
    T, V, mc = hubbard(2, 2, True)
    T2 = T.copy()
    T2[0::2, 0::2] *= 1.3                       # ↑ hops differently from ↓: H no longer commutes with S^±
    groups = su2.tensor_groups(T2, V, 2)
    # the hopping sits in the complementary operators S^A_p of F1/F1h: their two spin components no longer form a doublet
    assert max(su2.tensor_defect(g.T, g.k2, 2) for g in groups if g.family in ("F1", "F1h")) > 1e-3
    # the annihilation doublet is (c_↓, −c_↑): without the minus sign it is no tensor
    a = fock.annihilators(4)
    assert su2.tensor_defect({+1: a[1], -1: -a[0]}, 1, 2) < 1e-14
    assert su2.tensor_defect({+1: a[1], -1: a[0]}, 1, 2) > 0.5


@pytest.mark.parametrize("tS,tS2,k2", [(0, 1, 1), (1, 0, 1), (1, 2, 1), (2, 2, 2), (2, 0, 2), (3, 1, 2), (3, 3, 0), (4, 2, 2), (1, 1, 2)])
def test_recoupling_singlet_equals_its_closed_form(tS, tS2, k2):
    """With the Wigner–Eckart convention of this module the singlet recoupling sum collapses to
    √((2S′+1)/(2S+1)) (a 6j symbol with a zero argument) — the form the library's host code uses."""
    assert abs(su2.recoupling_singlet(tS, tS2, k2) - np.sqrt((tS2 + 1) / (tS + 1))) < 1e-13


def singlet_spectrum_from_S2(T, V, n_sites, N):
    """Eigenvalues of H inside the null space of S² with N particles — uses only the operator S²."""
    Sp, Sm, Sz, Nop = su2.spin_operators(n_sites)
    occ = fock.occupations(2 * n_sites)
    idx = np.flatnonzero((occ[:, 0::2].sum(1) == N // 2) & (occ[:, 1::2].sum(1) == N // 2))       # S_z = 0
    S2 = (Sz @ Sz + 0.5 * (Sp @ Sm + Sm @ Sp)).toarray()[np.ix_(idx, idx)]
    B = scipy.linalg.null_space(S2, rcond=1e-10)
    H = fock.hamiltonian(T, V).toarray()[np.ix_(idx, idx)]
    return np.linalg.eigvalsh(B.T @ H @ B)


@pytest.mark.parametrize("R,Cn,nA,rotated,keep", [(2, 2, 2, False, None), (2, 2, 2, True, None), (2, 2, 1, True, None),
                                                   (2, 3, 3, True, None), (2, 3, 2, True, None), (2, 3, 3, True, 0.6)])
def test_method_equals_definition_and_singlet_spectrum(R, Cn, nA, rotated, keep):
    T, V, mc = hubbard(R, Cn, rotated)
    n = R * Cn
    pb, multA, multB, groups, defects = su2.reduced_problem(T, V, nA, n, keep=keep, seed=5)
    assert defects["tensor_A"] < 1e-11 and defects["tensor_B"] < 1e-11
    assert defects["wigner_eckart"] < 1e-11                       # the quotient is the same for every (M, q)
    C = su2.singlet_isometry(multA, multB, n)
    assert np.abs(C.T @ C - np.eye(C.shape[1])).max() < 1e-12
    H = fock.hamiltonian(T, V)
    H_def = C.T @ (H @ C)                                          # the definition
    H_met = heff.dense_heff(pb)                                    # Σ scalar · L_red ⊗ R_red, blockwise
    assert H_met.shape == H_def.shape
    assert np.abs(H_met - H_def).max() < 1e-11 * max(1.0, np.abs(H_def).max())
    # σ through the blockwise tier with a random ψ
    rng = np.random.default_rng(3)
    pb.psi = {(a, b): rng.normal(size=(pb.sectors_A[a][1], pb.sectors_B[b][1])) for (a, b) in pb.psi_blocks()}
    sig = heff.sigma_blockwise(pb)
    x = heff.psi_to_vec(pb)
    assert np.abs(heff.psi_to_vec(pb, sig) - H_def @ x).max() < 1e-11 * np.abs(H_def @ x).max()
    if keep is None:
        ev = np.linalg.eigvalsh(H_def)
        ref = singlet_spectrum_from_S2(T, V, n, n)
        assert len(ev) == len(ref)                                 # number of singlets
        assert np.abs(ev - ref).max() < 1e-10
        # fewer states than U(1): "D stands for the number of renormalized multiplets"
        assert sum(d for _, d in pb.sectors_A) < 4 ** nA
    else:
        assert np.linalg.eigvalsh(H_met)[0] >= singlet_spectrum_from_S2(T, V, n, n)[0] - 1e-10     # variational


def test_hubbard_dimer_singlet_energy_closed_form():
    """Two sites, one per half: the three-multiplet dimer of tests/_su2.py, now derived instead of typed in;
    E0 = (U − √(U² + 16t²))/2 (tests/golden/closed_forms.txt)."""
    T, V, mc = lattice.hubbard_tV(None, 1.0, 4.0, bonds=[(0, 1)], n_sites=2)
    pb, *_ = su2.reduced_problem(T, V, 1, 2)
    assert [d for _, d in pb.sectors_A] == [1, 1, 1]
    E = np.linalg.eigvalsh(heff.dense_heff(pb))
    assert abs(E[0] - (4.0 - np.sqrt(16.0 + 16.0)) / 2) < 1e-13
