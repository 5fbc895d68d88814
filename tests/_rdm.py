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


# ---- two-particle reduced density matrix ("one- and two-body reduced density matrices";
#      the two-mode entropies of the mode optimisation need it) ----
def split_string(string, n_A):
    """A product of creators / annihilators  o_1 o_2 … o_m  (``string`` = [(mode, dagger)], modes of A are
    < n_A) rewritten as  sign · (A-operators in their order) · (B-operators in their order).

    Operators on different modes anticommute, so every B-operator that stands left of an A-operator costs
    one factor −1 when the A-operator is moved past it.  With the halves' own Jordan–Wigner strings
     the reordered product is  (Ã · P_A^π) ⊗ B̃ ,  π = number of B-operators mod 2."""
    sign, seen_B = 1.0, 0
    part_A, part_B = [], []
    for mode, dagger in string:
        if mode < n_A:
            part_A.append((mode, dagger))
            if seen_B & 1:
                sign = -sign
        else:
            part_B.append((mode - n_A, dagger))
            seen_B += 1
    return sign, part_A, part_B


def string_pairs(d, space, strings):
    """(Problem without ψ, kept) for a list of operator strings: one operator pair per string that conserves
    the charges (the others have expectation value 0 by symmetry and get no pair); ``kept`` = their indices."""
    n_A, n_B = space.A.n_modes, space.B.n_modes
    a, b = fock.annihilators(n_A), fock.annihilators(n_B)
    mc = d.mc
    nc = mc.shape[1]
    PhiA, PhiB = space.A.Phi, space.B.Phi
    pb = Problem(nc, list(space.sectors_A), list(space.sectors_B), tuple(space.target), name="strings")
    kept = []

    def shift(part, offset):
        dq = [0] * nc
        for mode, dagger in part:
            for c in range(nc):
                dq[c] += int(mc[mode + offset][c]) * (1 if dagger else -1)
        return tuple(dq)

    def product(part, ann):
        M = np.eye(ann[0].shape[0])
        for mode, dagger in part:
            M = M @ (ann[mode].T if dagger else ann[mode])
        return M

    def add_op(half, part, parity):
        Phi, sectors, ann, off = (PhiA, space.sectors_A, a, 0) if half == "A" else (PhiB, space.sectors_B, b, n_A)
        dq = shift(part, off)
        pb.ops.append({"half": half, "dq": dq, "parity": parity,
                       "blocks": _cut_blocks(Phi.T @ (product(part, ann) @ Phi), sectors, dq)})
        return len(pb.ops) - 1

    for idx, string in enumerate(strings):
        sign, part_A, part_B = split_string(string, n_A)
        if any(x + y != 0 for x, y in zip(shift(part_A, 0), shift(part_B, n_A))):
            continue
        parity = len(part_B) & 1
        assert (len(part_A) & 1) == parity       # charge conservation makes both halves odd or both even
        L = add_op("A", part_A, parity) if part_A else None
        R = add_op("B", part_B, parity) if part_B else None
        pb.terms.append((L, R, sign, False, False))
        kept.append(idx)
    return pb, kept


def rdm2_strings(n):
    """Labels (i, j, k, l), i < j, k < l, and the strings c†_i c†_j c_k c_l of Γ_ijkl = ⟨c†_i c†_j c_k c_l⟩;
    the other elements follow from Γ_ijkl = −Γ_jikl = −Γ_ijlk."""
    pairs = [(i, j) for i in range(n) for j in range(i + 1, n)]
    labels = [(i, j, k, l) for (i, j) in pairs for (k, l) in pairs]
    return labels, [[(i, True), (j, True), (k, False), (l, False)] for (i, j, k, l) in labels]


def rdm2_fock(d, space, x, labels):
    """Γ_ijkl = ⟨Ψ| c†_i c†_j c_k c_l |Ψ⟩ with Ψ = P x in the full Fock space (the definition), per label."""
    n = d.n
    c = fock.annihilators(n)
    psi = np.zeros(2 ** n)
    psi[d.rows] = dmrg.projector(space, d.rows) @ x
    return np.array([float(psi @ (c[i].T @ (c[j].T @ (c[k] @ (c[l] @ psi))))) for (i, j, k, l) in labels])
