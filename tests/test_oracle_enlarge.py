"""Pins for the block-enlargement half of the renormalisation step:
`oracle.renorm.enlarge_dense` (Σ coef (X P^π) ⊗ y with explicit Kronecker products) evaluated on the
product lists of the library's host builder (`paper_2311_14106_b200.blockops`, host logic) must equal
the DEFINITION of the next bond's block operators, Φ_{A′}† O Φ_{A′}, built from Fock-space matrices
(`oracle.terms.complementary_terms` on A′, projected with the explicit DMRG basis of `oracle.dmrg`).
This pins every sign, ½ and index of the S^{A′}_p accumulation and of the H_{A′} coupling terms."""
import numpy as np
import pytest

from oracle import lattice, dmrg, terms as oterms, renorm
from paper_2311_14106_b200 import blockops


def spinless_3x3(D, rotated=True):
    T, V, mc = lattice.spinless_tV(3)
    if rotated:
        T, V = lattice.rotate(T, V, lattice.rotation_matrix(9, seed=3))
    return T, V, mc, [[i] for i in range(9)], (4,), D


def hubbard_ring(D):
    bonds = [(0, 1), (1, 2), (2, 3), (3, 0)]
    T, V, mc = lattice.hubbard_tV(None, 1.0, 4.0, bonds=bonds, n_sites=4)
    T, V = lattice.rotate(T, V, lattice.spin_rotation(lattice.rotation_matrix(4, seed=4, std=0.3)))
    return T, V, mc, [[0, 1], [2, 3], [4, 5], [6, 7]], (2, 2), D


def fock_operator_set(T, V, mc, n_A):
    """{key: sparse operator on the Fock space of modes 0..n_A−1}: the left-block set, from the oracle's
    regrouping of Eq. (1) across the cut after mode n_A−1 (prune=False keeps every pair)."""
    out = {}
    for t in oterms.complementary_terms(T, V, n_A, mc, prune=False):
        if t.family == "F0" and t.label == ("A",):
            out[("H",)] = t.X
        elif t.family == "F1":
            out[("S", t.label[0])] = t.X
        elif t.family == "F2":
            out[("c+", t.label[0])] = t.X
        elif t.family == "F3":
            out[("c+c+",) + tuple(t.label)] = t.X
        elif t.family == "F4" and t.label[0] <= t.label[1]:
            out[("c+c",) + tuple(t.label)] = t.X
    return out


def bond_step(make, bond):
    """DMRG warmed up to `bond`, one more step to the right: returns what the enlargement test needs."""
    T, V, mc, site_modes, target, D = make
    d = dmrg.SimpleDMRG(T, V, mc, site_modes, target, D=D, seed=2)
    d.warmup_to(bond)
    d.step(bond, +1)                                   # sets d.L[bond + 1]: the kept basis of A
    kept, sectors_K = dmrg.sector_major(d.L[bond + 1])
    A = [m for s in site_modes[:bond + 1] for m in s]
    S = list(site_modes[bond + 1])
    right = [m for s in site_modes[bond + 2:] for m in s]
    return d, kept, sectors_K, A, S, right


@pytest.mark.parametrize("make,bond", [(spinless_3x3(64), 3), (spinless_3x3(5), 3), (spinless_3x3(6, rotated=False), 4),
                                       (hubbard_ring(6), 0), (hubbard_ring(16), 1)])
def test_builder_lists_reproduce_the_definition(make, bond):
    T, V, mc = make[0], make[1], make[2]
    d, kept, sectors_K, A, S, right = bond_step(make, bond)
    n_A, n_Ap = len(A), len(A) + len(S)
    # kept operators of A (dense, in the kept basis): Φ† X Φ from Fock space
    XA = fock_operator_set(T, V, mc, n_A)
    keptops = {k: kept.Phi.T @ (X @ kept.Phi) for k, X in XA.items()}
    assert set(keptops) == set(blockops.left_block_keys(A, S + right))
    site, lists = blockops.enlarge_left_lists(T, V, mc, A, S, right)
    # definition on A′
    Ap, sectors_E = dmrg.sector_major(dmrg.kron_basis(kept, dmrg.site_basis(d.mc[S])))
    perm, sectors_E2 = renorm.enlarged_order(sectors_K, site.charges.tolist())
    assert sectors_E2 == sectors_E                                     # same sector-major ordering of A′
    XAp = fock_operator_set(T, V, mc, n_Ap)
    assert set(lists) == set(XAp) == set(blockops.left_block_keys(A + S, right))
    worst = 0.0
    for key, plist in lists.items():
        terms = [(None if k is None else (keptops[k].T if tr else keptops[k]), y, 1.0, pi) for (k, tr, y, pi) in plist]
        got = renorm.enlarge_dense(terms, sectors_K, site.charges.tolist())
        ref = Ap.Phi.T @ (XAp[key] @ Ap.Phi)
        scale = max(1.0, np.abs(ref).max())
        worst = max(worst, np.abs(got - ref).max() / scale)
        assert np.abs(got - ref).max() <= 1e-12 * scale, key
        dq, parity = blockops.operator_spec(key, mc)
        assert parity == (1 if key[0] in ("S", "c+") else 0)
    assert worst <= 1e-12


def test_a_wrong_sign_is_caught():
    """Flipping the sign rule of one family breaks the identity (the pin is sensitive)."""
    make = spinless_3x3(64)
    T, V, mc = make[0], make[1], make[2]
    d, kept, sectors_K, A, S, right = bond_step(make, 3)
    XA = fock_operator_set(T, V, mc, len(A))
    keptops = {k: kept.Phi.T @ (X @ kept.Phi) for k, X in XA.items()}
    site, lists = blockops.enlarge_left_lists(T, V, mc, A, S, right)
    Ap, _ = dmrg.sector_major(dmrg.kron_basis(kept, dmrg.site_basis(d.mc[S])))
    XAp = fock_operator_set(T, V, mc, len(A) + len(S))
    key = ("S", right[0])
    ref = Ap.Phi.T @ (XAp[key] @ Ap.Phi)
    for drop_parity in (False, True):
        terms = [(None if k is None else (keptops[k].T if tr else keptops[k]), y, 1.0, 0 if drop_parity else pi)
                 for (k, tr, y, pi) in lists[key]]
        err = np.abs(renorm.enlarge_dense(terms, sectors_K, site.charges.tolist()) - ref).max()
        assert (err > 1e-3) == drop_parity


# ---- right block: B′ = site ⊗ kept B, with the S, P, Q accumulations --------------------------------
def fock_right_set(T, V, mc, n_A):
    """{key: sparse operator on the Fock space of modes n_A..n−1 (B's own JW basis)}: the right-block set."""
    out = {}
    for t in oterms.complementary_terms(T, V, n_A, mc, prune=False):
        if t.family == "F0" and t.label == ("B",):
            out[("H",)] = t.Y
        elif t.family == "F1":
            out[("c+", t.label[0])] = t.Y
        elif t.family == "F2":
            out[("S", t.label[0])] = t.Y
        elif t.family == "F3":
            out[("P",) + tuple(t.label)] = t.Y
        elif t.family == "F4" and t.label[0] <= t.label[1]:
            out[("Q",) + tuple(t.label)] = t.Y
    return out


@pytest.mark.parametrize("make,bond", [(spinless_3x3(64), 4), (spinless_3x3(5), 4), (spinless_3x3(6, rotated=False), 3),
                                       (hubbard_ring(6), 2), (hubbard_ring(16), 1)])
def test_right_block_lists_reproduce_the_definition(make, bond):
    T, V, mc, site_modes, target, D = make
    d = dmrg.SimpleDMRG(T, V, mc, site_modes, target, D=D, seed=2)
    d.warmup_to(bond)
    d.step(bond, -1)                                   # sets d.R[bond + 1]: the kept basis of B = site(bond+1) ∪ …
    kept, sectors_K = dmrg.sector_major(d.R[bond + 1])      # a relabelling: R's columns come in descending charge order
    left = [m for s in site_modes[:bond] for m in s]
    S = list(site_modes[bond])
    B = [m for s in site_modes[bond + 1:] for m in s]
    n_A = len(left) + len(S)
    YB = fock_right_set(T, V, mc, n_A)
    keptops = {k: kept.Phi.T @ (Y @ kept.Phi) for k, Y in YB.items()}
    assert set(keptops) == set(blockops.right_block_keys(B, left + S))
    site, lists = blockops.enlarge_right_lists(T, V, mc, left, S, B)
    Bp, sectors_E = dmrg.sector_major(dmrg.kron_basis(dmrg.site_basis(d.mc[S]), kept))
    perm, sectors_E2 = renorm.enlarged_order_right(sectors_K, site.charges.tolist())
    assert sectors_E2 == sectors_E
    YBp = fock_right_set(T, V, mc, len(left))
    assert set(lists) == set(YBp) == set(blockops.right_block_keys(S + B, left))
    for key, plist in lists.items():
        terms = [(None if k is None else (keptops[k].T if tr else keptops[k]), y, 1.0, blockops.right_key_parity(k))
                 for (k, tr, y, odd) in plist]
        got = renorm.enlarge_dense_right(terms, sectors_K, site.charges.tolist(), site.parity)
        ref = Bp.Phi.T @ (YBp[key] @ Bp.Phi)
        scale = max(1.0, np.abs(ref).max())
        assert np.abs(got - ref).max() <= 1e-12 * scale, key
