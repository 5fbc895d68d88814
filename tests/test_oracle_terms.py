"""Pins for oracle/terms.py: the complementary-operator regrouping of Eq. (1)
 must reproduce the Fock-space Hamiltonian exactly."""
import numpy as np
import pytest

from oracle import fock, lattice, terms


@pytest.mark.parametrize("n,n_A", [(6, 3), (6, 2), (6, 4), (5, 1), (7, 3)])
def test_regrouping_reproduces_H_random_nonhermitian(n, n_A):
    rng = np.random.default_rng(100 + n * 10 + n_A)
    T = rng.normal(size=(n, n))
    V = rng.normal(size=(n, n, n, n))       # no symmetry at all: every family is exercised on its own
    H = fock.hamiltonian(T, V)
    tm = terms.complementary_terms(T, V, n_A, np.ones((n, 1)))
    n_B = n - n_A
    assert len(tm) == 2 + 2 * n_B + 2 * n_A + n_A * (n_A - 1) + n_A * n_A
    assert abs(H - terms.assemble(tm, n_A, n_B)).max() < 1e-12


def test_each_family_is_needed():
    # dropping any one family must break the identity (guards against a family silently being zero)
    rng = np.random.default_rng(5)
    n, n_A = 6, 3
    T = rng.normal(size=(n, n)); V = rng.normal(size=(n, n, n, n))
    H = fock.hamiltonian(T, V)
    tm = terms.complementary_terms(T, V, n_A, np.ones((n, 1)))
    for fam in ("F0", "F1", "F1h", "F2", "F2h", "F3", "F3h", "F4"):
        rest = [t for t in tm if t.family != fam]
        assert abs(H - terms.assemble(rest, n_A, n - n_A)).max() > 1e-3, fam


def test_sign_of_fermionic_families_matters():
    rng = np.random.default_rng(6)
    n, n_A = 6, 3
    T = rng.normal(size=(n, n)); V = rng.normal(size=(n, n, n, n))
    H = fock.hamiltonian(T, V)
    tm = terms.complementary_terms(T, V, n_A, np.ones((n, 1)))
    for t in tm:
        if t.family == "F1":
            t.coef = +1.0        # the wrong sign
    assert abs(H - terms.assemble(tm, n_A, n - n_A)).max() > 1e-3
    # ... and so does the parity string on the A factor
    tm = terms.complementary_terms(T, V, n_A, np.ones((n, 1)))
    for t in tm:
        t.parity = 0
    assert abs(H - terms.assemble(tm, n_A, n - n_A)).max() > 1e-3


def test_real_space_term_counts():
    # 4×4 real space, middle cut: K = 2 + 16 hopping S-terms + 8 n_p ⊗ Q_pp = 26
    T, V, mc = lattice.spinless_tV(4)
    tm = terms.complementary_terms(T, V, 8, mc)
    fams = [t.family for t in tm]
    assert len(tm) == 26 and fams.count("F1") == 8 and fams.count("F1h") == 8 and fams.count("F4") == 8
    H = fock.hamiltonian(T, V)
    # 16 modes: compare on the N=8 sector only (the full 65536² difference is sparse anyway)
    idx = fock.sector_indices(16, mc, (8,))
    D = fock.restrict(H - terms.assemble(tm, 8, 8), idx)
    assert abs(D).max() < 1e-12


def test_hermitian_partner_structure_and_shifts():
    T, V, mc = lattice.spinless_tV(3)
    U = lattice.rotation_matrix(9, seed=3)
    T, V = lattice.rotate(T, V, U)
    n_A = 4
    tm = terms.complementary_terms(T, V, n_A, mc)
    by = {(t.family, t.label): t for t in tm}
    for (fam, lab), t in by.items():
        if fam == "F1":
            h = by[("F1h", lab)]
            assert abs(h.X - t.X.T).max() < 1e-12 and abs(h.Y - t.Y.T).max() < 1e-12
            assert h.coef == -t.coef          # odd pair: h.c. partner carries −c
        if fam == "F2":
            h = by[("F2h", lab)]
            assert abs(h.X - t.X.T).max() < 1e-12 and abs(h.Y - t.Y.T).max() < 1e-12
            assert h.coef == -t.coef
        if fam == "F3":
            h = by[("F3h", lab)]
            assert abs(h.X - t.X.T).max() < 1e-12 and abs(h.Y - t.Y.T).max() < 1e-12
            assert h.coef == t.coef
        if fam == "F4" and lab[0] != lab[1]:
            h = by[("F4", (lab[1], lab[0]))]
            assert abs(h.X - t.X.T).max() < 1e-12 and abs(h.Y - t.Y.T).max() < 1e-12
    # charge shifts: X maps N → N + dq_A on A, Y maps N → N − dq_A on B
    NA = fock.occupations(n_A).sum(axis=1)
    NB = fock.occupations(9 - n_A).sum(axis=1)
    for t in tm:
        r, c = t.X.nonzero()
        assert np.all(NA[r] - NA[c] == t.dq_A[0])
        r, c = t.Y.nonzero()
        assert np.all(NB[r] - NB[c] == -t.dq_A[0])
        assert t.parity == abs(t.dq_A[0]) % 2


def test_hubbard_two_charge_regrouping():
    T, V, mc = lattice.hubbard_tV(None, 1.0, 4.0, bonds=[(0, 1), (1, 2), (2, 0)], n_sites=3)
    U2 = lattice.spin_rotation(lattice.rotation_matrix(3, seed=4, std=0.4))
    T, V = lattice.rotate(T, V, U2)
    n_A = 2    # cut inside nothing: site 0 | sites 1,2
    tm = terms.complementary_terms(T, V, n_A, mc, prune=False)
    H = fock.hamiltonian(T, V)
    assert abs(H - terms.assemble(tm, n_A, 6 - n_A)).max() < 1e-12
    qA = fock.charges_of_states(n_A, mc[:n_A])
    for t in tm:
        r, c = t.X.nonzero()
        assert np.all(qA[r] - qA[c] == np.array(t.dq_A))
