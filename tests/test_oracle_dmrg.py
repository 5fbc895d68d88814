"""Pins for oracle/dmrg.py, export.py, davidson.py (T1, T1x): the definition
H_eff = P†HP against the exported block lists, DMRG against exact diagonalisation."""
import numpy as np
import pytest

from oracle import fock, lattice, dmrg, heff, export, davidson
from _util import golden_table


@pytest.fixture(scope="module")
def dmrg_3x3():
    T, V, mc = lattice.spinless_tV(3)
    d = dmrg.SimpleDMRG(T, V, mc, [[i] for i in range(9)], (4,), D=64, seed=1)
    d.warmup_to(4)
    return d


def test_dmrg_untruncated_equals_ed(dmrg_3x3):
    g = golden_table("ed_energies.txt")
    # D = 64 exceeds every Schmidt rank of the 126-dim N=4 sector: DMRG is exact
    assert abs(dmrg_3x3.energies[-1] - float(g["spinless_3x3_N4"])) < 1e-10


def test_dmrg_truncated_is_variational():
    g = golden_table("ed_energies.txt")
    T, V, mc = lattice.spinless_tV(3)
    d = dmrg.SimpleDMRG(T, V, mc, [[i] for i in range(9)], (4,), D=4, seed=1)
    d.warmup_to(4)
    assert all(e >= float(g["spinless_3x3_N4"]) - 1e-12 for e in d.energies)
    assert d.energies[-1] > float(g["spinless_3x3_N4"]) + 1e-6


def test_bases_are_isometries_with_definite_charge(dmrg_3x3):
    for b in list(dmrg_3x3.L.values()) + list(dmrg_3x3.R.values()):
        assert np.abs(b.Phi.T @ b.Phi - np.eye(b.Phi.shape[1])).max() < 1e-12
        occ = fock.occupations(b.n_modes).sum(axis=1)
        for col in range(b.Phi.shape[1]):
            support = np.abs(b.Phi[:, col]) > 1e-12
            assert np.all(occ[support] == b.q[col, 0])


@pytest.mark.parametrize("rotated,D", [(False, 64), (True, 6), (False, 5)])
def test_exported_blocks_reproduce_PHP(rotated, D):
    """T1 (definition) vs T2 and T3 (block lists), truncated and untruncated bases,
    real-space (pruned, K small) and rotated (dense, all families)."""
    T, V, mc = lattice.spinless_tV(3)
    if rotated:
        T, V = lattice.rotate(T, V, lattice.rotation_matrix(9, seed=3))
    d = dmrg.SimpleDMRG(T, V, mc, [[i] for i in range(9)], (4,), D=D, seed=2)
    d.warmup_to(4)
    space = d.space_at(4)
    Heff, P = d.heff_at(space)
    x = d.guess_at(space, P)
    for pairs in (True, False):
        pb = export.export_bond(d, space, use_transpose_pairs=pairs)
        pb.psi = dmrg.vec_to_blocks(space, x)
        Hd = heff.dense_heff(pb)
        assert np.abs(Hd - Heff).max() < 1e-12
        s3 = heff.psi_to_vec(pb, heff.sigma_blockwise(pb))
        assert np.abs(s3 - Heff @ x).max() < 1e-12
        if rotated:
            n_A = space.A.n_modes
            assert len(pb.terms) == 2 + 2 * (9 - n_A) + 2 * n_A + n_A * (n_A - 1) + n_A * n_A
            assert any(t[3] for t in pb.terms) == pairs


def test_hubbard_two_charge_export():
    bonds = [(0, 1), (1, 2), (2, 3), (3, 0)]
    T, V, mc = lattice.hubbard_tV(None, 1.0, 4.0, bonds=bonds, n_sites=4)
    U2 = lattice.spin_rotation(lattice.rotation_matrix(4, seed=4, std=0.3))
    T, V = lattice.rotate(T, V, U2)
    d = dmrg.SimpleDMRG(T, V, mc, [[0, 1], [2, 3], [4, 5], [6, 7]], (2, 2), D=6, seed=3)
    d.warmup_to(1)
    space = d.space_at(1)
    Heff, P = d.heff_at(space)
    x = d.guess_at(space, P)
    pb = export.export_bond(d, space)
    pb.psi = dmrg.vec_to_blocks(space, x)
    assert np.abs(heff.dense_heff(pb) - Heff).max() < 1e-12
    assert np.abs(heff.psi_to_vec(pb, heff.sigma_blockwise(pb)) - Heff @ x).max() < 1e-12
    E_ed = fock.ground_energy(T, V, mc, (2, 2))
    assert d.energies[-1] >= E_ed - 1e-12


def test_davidson_matches_dense_eigh():
    import workloads as wlmod
    wl = wlmod.lattice_workload("spinless", 5, 24, seed=3)
    pb = heff.problem_from_workload(wl)
    H = heff.dense_heff(pb)
    dg = heff.psi_to_vec(pb, heff.diagonal_blockwise(pb))
    x0 = heff.psi_to_vec(pb)
    hist = []
    theta, x, n_apply = davidson.davidson(lambda v: H @ v, dg, x0, tol=1e-10, history=hist)
    E = np.linalg.eigvalsh(H)[0]
    assert abs(theta - E) < 1e-9 * max(1.0, abs(E))
    th = [h[0] for h in hist]
    assert all(b <= a + 1e-12 for a, b in zip(th, th[1:]))      # Ritz values never increase
    assert np.linalg.norm(H @ x - theta * x) < 1e-9
    assert n_apply == len(hist)


def test_davidson_restart_path():
    rng = np.random.default_rng(0)
    n = 200
    A = rng.normal(size=(n, n)); A = A + A.T + np.diag(np.arange(n) * 0.5)
    theta, x, n_apply = davidson.davidson(lambda v: A @ v, np.diag(A).copy(), rng.normal(size=n),
                                          tol=1e-9, m_max=4, max_iter=2000)
    assert abs(theta - np.linalg.eigvalsh(A)[0]) < 1e-9


@pytest.mark.slow
def test_config1_D256_equals_ed():
    """BASELINE.json config 1 oracle check: D=256 is exact by dimension counting."""
    g = golden_table("ed_energies.txt")
    T, V, mc = lattice.spinless_tV(4)
    d = dmrg.SimpleDMRG(T, V, mc, [[i] for i in range(16)], (8,), D=256, seed=1)
    d.sweep_right(0, 8)
    assert abs(d.energies[-1] - float(g["spinless_4x4_N8"])) < 1e-9
