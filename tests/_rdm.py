"""Test helper: the operator-pair list whose expectation values are the one-particle reduced density
matrix γ_ij = ⟨c†_i c_j⟩ at a DMRG bond of the oracle, and its Fock-space definition."""
import numpy as np

from oracle import fock, dmrg
from oracle.export import _cut_blocks
from oracle.heff import Problem


def rdm_pairs(d, space):
    """(Problem without ψ, [(i, j)] per term) for i ≤ j over all modes; A's modes precede B's, so
    c†_i c_j = (c̃†_i c̃_j) ⊗ 1, 1 ⊗ (c̃†_i c̃_j) or (c̃†_i P) ⊗ c̃_j — all with coefficient +1."""
    n_A, n_B = space.A.n_modes, space.B.n_modes
    a, b = fock.annihilators(n_A), fock.annihilators(n_B)
    mc = d.mc
    q = lambda p: tuple(int(x) for x in mc[p])
    sub = lambda s, t: tuple(x - y for x, y in zip(s, t))
    neg = lambda t: tuple(-x for x in t)
    PhiA, PhiB = space.A.Phi, space.B.Phi
    pb = Problem(mc.shape[1], list(space.sectors_A), list(space.sectors_B), tuple(space.target), name="rdm")
    labels = []

    def add_op(half, M, dq, parity):
        Phi, sectors = (PhiA, space.sectors_A) if half == "A" else (PhiB, space.sectors_B)
        pb.ops.append({"half": half, "dq": dq, "parity": parity, "blocks": _cut_blocks(Phi.T @ (M @ Phi), sectors, dq)})
        return len(pb.ops) - 1

    for i in range(n_A + n_B):
        for j in range(i, n_A + n_B):
            if q(i) != q(j):
                continue            # c†_i c_j changes a conserved charge: γ_ij = 0 by symmetry, no operator pair
            if j < n_A:
                L, R = add_op("A", a[i].T @ a[j], sub(q(i), q(j)), 0), None
            elif i >= n_A:
                L, R = None, add_op("B", b[i - n_A].T @ b[j - n_A], sub(q(i), q(j)), 0)
            else:
                L, R = add_op("A", a[i].T, q(i), 1), add_op("B", b[j - n_A], neg(q(j)), 1)
            pb.terms.append((L, R, 1.0, False, False))
            labels.append((i, j))
    return pb, labels


def rdm_fock(d, space, x):
    """γ_ij = ⟨Ψ| c†_i c_j |Ψ⟩ with Ψ = P x in the full Fock space (the definition)."""
    n = d.n
    c = fock.annihilators(n)
    psi = np.zeros(2 ** n)
    psi[d.rows] = dmrg.projector(space, d.rows) @ x
    cpsi = [ci @ psi for ci in c]
    return np.array([[float(cpsi[i] @ cpsi[j]) for j in range(n)] for i in range(n)])
