"""Pins for oracle/heff.py (T2 Kronecker, T3 blockwise) on seeded synthetic workloads."""
import numpy as np
import pytest

import workloads as wlmod
from oracle import heff


def small_config2():
    return wlmod.synthetic_config2(M=64, n_q=9, K=32, seed=2, width2=8.0)


def small_spinless(keep=None):
    return wlmod.lattice_workload("spinless", 5, 24, seed=3, keep=keep)


def small_hubbard():
    thin = lambda fam, i: fam in ("F1", "F2") or i % 3 == 0
    return wlmod.lattice_workload("hubbard", 2, 14, seed=4, keep=thin)


def rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def test_restricted_kron_equals_full_kron():
    wl = wlmod.synthetic_config2(M=12, n_q=5, K=6, seed=7, width2=4.0)
    pb = heff.problem_from_workload(wl)
    full = heff.full_kron_heff(pb)
    ia, ib = heff.allowed_pairs(pb)
    MB = wl.M_B
    lin = ia * MB + ib
    assert np.abs(full[np.ix_(lin, lin)] - heff.dense_heff(pb)).max() < 1e-13
    # charge conservation: H_eff maps the target sector into itself
    other = np.setdiff1d(np.arange(full.shape[0]), lin)
    assert np.abs(full[np.ix_(other, lin)]).max() == 0.0
    # and vec(ψ) row-major (a major) reproduces the matrix form L ψ Rᵀ
    psi = heff.densify_psi(pb)
    sig = (full @ psi.reshape(-1)).reshape(psi.shape)
    got = heff.densify_psi(pb, heff.sigma_dense(pb))
    assert np.abs(sig - got).max() < 1e-12


@pytest.mark.parametrize("make", [small_config2, small_spinless, small_hubbard])
def test_T3_matches_T2(make):
    pb = heff.problem_from_workload(make())
    s2 = heff.psi_to_vec(pb, heff.sigma_dense(pb))
    s3 = heff.psi_to_vec(pb, heff.sigma_blockwise(pb))
    assert np.abs(s2).max() > 0
    assert rel(s3, s2) < 1e-13


def test_T3_library_product_vs_explicit_loops():
    wl = wlmod.synthetic_config2(M=24, n_q=7, K=8, seed=5, width2=6.0)
    pb = heff.problem_from_workload(wl)
    a = heff.psi_to_vec(pb, heff.sigma_blockwise(pb, naive=True))
    b = heff.psi_to_vec(pb, heff.sigma_blockwise(pb))
    assert rel(a, b) < 1e-13


@pytest.mark.parametrize("make", [small_spinless, small_hubbard])
def test_hermitian_construction_gives_symmetric_heff(make):
    """Pins the transpose-flag pairing and the sign rule (odd h.c. partner ↔ −c, sign tied
    to the *input* A charge): any slip makes H_eff non-symmetric."""
    pb = heff.problem_from_workload(make())
    H = heff.dense_heff(pb)
    assert np.abs(H).max() > 0.1
    assert np.abs(H - H.T).max() < 1e-12 * np.abs(H).max()
    # flipping one partner coefficient breaks it
    k = next(i for i, t in enumerate(pb.terms) if t[3] and pb.ops[t[0]]["parity"] == 1)
    L, R, c, tl, tr = pb.terms[k]
    pb.terms[k] = (L, R, -c, tl, tr)
    H2 = heff.dense_heff(pb)
    assert np.abs(H2 - H2.T).max() > 1e-3


def test_config2_is_not_symmetric():
    H = heff.dense_heff(heff.problem_from_workload(small_config2()))
    assert np.abs(H - H.T).max() > 1e-3       # r15: matvec-only workload


def test_block_support_single_input_block():
    wl = small_config2()
    pb = heff.problem_from_workload(wl)
    blocks = pb.psi_blocks()
    src = blocks[len(blocks) // 2]
    psi = {k: (v if k == src else np.zeros_like(v)) for k, v in pb.psi.items()}
    sig = heff.sigma_blockwise(pb, psi)
    shifts = {wl.ops[t.L].dq[0] for t in wl.terms}
    for (ai, bi), blk in sig.items():
        d = pb.sectors_A[ai][0][0] - pb.sectors_A[src[0]][0][0]
        if np.abs(blk).max() > 0:
            assert d in shifts


def test_linearity_and_k_additivity():
    pb = heff.problem_from_workload(small_spinless())
    full = heff.psi_to_vec(pb, heff.sigma_blockwise(pb))
    terms = list(pb.terms)
    pb.terms = terms[:7]
    a = heff.psi_to_vec(pb, heff.sigma_blockwise(pb))
    pb.terms = terms[7:]
    b = heff.psi_to_vec(pb, heff.sigma_blockwise(pb))
    assert rel(a + b, full) < 1e-13


def test_diagonal_blockwise_vs_dense():
    for make in (small_spinless, small_hubbard, small_config2):
        pb = heff.problem_from_workload(make())
        d = heff.psi_to_vec(pb, heff.diagonal_blockwise(pb))
        assert np.abs(d - np.diag(heff.dense_heff(pb))).max() < 1e-12


def test_flops_alg_hand_count():
    # two sectors of dims (2,3) on A and (3,2) on B, one pair with shift +1/-1
    pb = heff.Problem(1, [((0,), 2), ((1,), 3)], [((0,), 3), ((1,), 2)], (1,))
    pb.ops = [{"half": "A", "dq": (1,), "parity": 1, "blocks": {(1, 0): np.ones((3, 2))}},
              {"half": "B", "dq": (-1,), "parity": 1, "blocks": {(0, 1): np.ones((3, 2))}}]
    pb.terms = [(0, 1, 1.0, False, False)]
    pb.psi = {(0, 1): np.ones((2, 2)), (1, 0): np.ones((3, 3))}
    # only input block (a=0,b=1): m=2,n=2 → output (1,0): m'=3,n'=3
    assert heff.flops_alg(pb) == min(2 * 3 * 2 * (2 + 3), 2 * 2 * 3 * (2 + 3))
    sig = heff.sigma_blockwise(pb)
    # L ψ Rᵀ with all-ones = 2·2 = 4 in every entry, sign (+) since N(q_a = 0) is even
    assert np.all(sig[(1, 0)] == 4.0) and np.all(sig[(0, 1)] == 0.0)


def test_fermionic_sign_uses_input_A_parity():
    pb = heff.Problem(1, [((0,), 1), ((1,), 1), ((2,), 1)], [((0,), 1), ((1,), 1), ((2,), 1)], (2,))
    pb.ops = [{"half": "A", "dq": (1,), "parity": 1, "blocks": {(1, 0): np.ones((1, 1)), (2, 1): np.ones((1, 1))}},
              {"half": "B", "dq": (-1,), "parity": 1, "blocks": {(0, 1): np.ones((1, 1)), (1, 2): np.ones((1, 1))}}]
    pb.terms = [(0, 1, 1.0, False, False)]
    pb.psi = {(0, 2): np.ones((1, 1)), (1, 1): np.ones((1, 1)), (2, 0): np.ones((1, 1))}
    sig = heff.sigma_blockwise(pb)
    assert sig[(1, 1)][0, 0] == +1.0      # from input a-sector N=0 (even)
    assert sig[(2, 0)][0, 0] == -1.0      # from input a-sector N=1 (odd)
    s2 = heff.sigma_dense(pb)
    assert s2[(1, 1)][0, 0] == +1.0 and s2[(2, 0)][0, 0] == -1.0


def test_block_coefficients_blockwise_vs_kronecker_and_su2_dimer():
    """The per-(pair, input block) scalar: T3 against T2 with random scalars incl.
    zeros, and the spin-singlet H_eff of the Hubbard dimer against its closed form."""
    import workloads as wlmod
    from _su2 import dimer_singlet_problem
    from _util import golden_table
    pb = heff.problem_from_workload(wlmod.lattice_workload("spinless", 5, 24, seed=3))
    rng = np.random.default_rng(5)
    pb.block_coef = {(k, blk): (0.0 if rng.random() < 0.2 else float(rng.normal())) for k in range(len(pb.terms))
                     for blk in pb.psi_blocks() if rng.random() < 0.7}
    s2, s3 = heff.sigma_dense(pb), heff.sigma_blockwise(pb)
    assert max(np.abs(s2[k] - s3[k]).max() for k in s2) < 1e-12
    plain = heff.problem_from_workload(wlmod.lattice_workload("spinless", 5, 24, seed=3))
    assert max(np.abs(heff.sigma_blockwise(plain)[k] - s3[k]).max() for k in s3) > 1e-3      # the scalars matter
    dim, H = dimer_singlet_problem()
    assert np.abs(heff.dense_heff(dim) - H).max() < 1e-14
    E0 = float(golden_table("closed_forms.txt")["hubbard_dimer_E0_U4"])
    assert abs(np.linalg.eigvalsh(heff.dense_heff(dim))[0] - E0) < 1e-12
