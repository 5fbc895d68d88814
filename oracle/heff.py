"""T2 / T3: σ = Σ_k c_k (L_k ⊗ R_k) ψ from block lists (BASELINE.json north_star;
SURVEY.md §8.0 for the exact formula, §8(c) tiers T2 and T3).

A `Problem` is what the GPU library consumes, as plain NumPy:
  sectors_A / sectors_B : [(charge tuple, dim)] of the enlarged blocks
  target                : total charge; ψ has a block (a, b) wherever q_a + q_b = target
  ops[i]                : {"half", "dq", "parity", "blocks": {(row_idx, col_idx): array}}
                          — block (row, col) maps column sector q to row sector q + dq
  terms[k]              : (L, R, coef, trans_L, trans_R); L or R None = identity;
                          trans_X means "use the transpose of the stored operator"
  psi                   : {(a_idx, b_idx): array}

Definition (the formula both tiers implement):
    σ = Σ_k c_k · (op_L(k) · P^{π_k}) ψ op_R(k)ᵀ ,   ψ ≡ matrix ψ[a, b],
    P = diag((−1)^{N(q_a)}) on the *input* A index, N(q) = Σ of the charge
    components (particle number), π_k = parity of the pair.
T2 writes it as the dense matrix Σ_k c_k kron(op_L P^π, op_R) restricted to the
allowed (a, b) pairs; T3 does it block by block with one dense product per
step.  T3 with BLAS products is also the timed CPU baseline of bench.py.
"""
from dataclasses import dataclass, field
import numpy as np


@dataclass
class Problem:
    n_charges: int
    sectors_A: list
    sectors_B: list
    target: tuple
    ops: list = field(default_factory=list)
    terms: list = field(default_factory=list)
    psi: dict = field(default_factory=dict)
    name: str = ""
    block_coef: dict = None      # optional {(k, (a_idx, b_idx)): scalar}: an extra factor of pair k on INPUT block (a, b)
                                 # — the per-block-pair recoupling scalar of SU(2)-adapted DMRG;
                                 # a missing key means 1, a zero removes the task

    def psi_blocks(self):
        idxB = {q: i for i, (q, _) in enumerate(self.sectors_B)}
        out = []
        for ai, (qa, da) in enumerate(self.sectors_A):
            qb = tuple(t - x for t, x in zip(self.target, qa))
            if qb in idxB and da > 0 and self.sectors_B[idxB[qb]][1] > 0:
                out.append((ai, idxB[qb]))
        return out


def problem_from_workload(wl, with_psi=True):
    """Materialise a (small) seeded workload of ``workloads`` on the host."""
    from workloads import fill_op_host, fill_psi_host
    ops = []
    for i, spec in enumerate(wl.ops):
        ops.append({"half": spec.half, "dq": tuple(spec.dq), "parity": spec.parity,
                    "blocks": fill_op_host(wl, i)})
    terms = [(t.L, t.R, t.coef, t.trans_L, t.trans_R) for t in wl.terms]
    psi = fill_psi_host(wl) if with_psi else {}
    return Problem(wl.n_charges, list(wl.sectors_A), list(wl.sectors_B), tuple(wl.target),
                   ops, terms, psi, wl.name)


def sector_offsets(sectors):
    off, o = [], 0
    for _, d in sectors:
        off.append(o)
        o += d
    return off, o


def sector_parity(q):
    """Fermion parity of a sector: particle number = sum of charge components."""
    return int(sum(q)) % 2


def densify_op(op, sectors, trans=False):
    """Dense M × M matrix of a stored operator (sector-major basis), optionally transposed."""
    off, M = sector_offsets(sectors)
    D = np.zeros((M, M))
    for (ri, ci), blk in op["blocks"].items():
        D[off[ri]:off[ri] + blk.shape[0], off[ci]:off[ci] + blk.shape[1]] = blk
    return D.T.copy() if trans else D


def densify_psi(pb, psi=None):
    offA, MA = sector_offsets(pb.sectors_A)
    offB, MB = sector_offsets(pb.sectors_B)
    X = np.zeros((MA, MB))
    for (ai, bi), blk in (pb.psi if psi is None else psi).items():
        X[offA[ai]:offA[ai] + blk.shape[0], offB[bi]:offB[bi] + blk.shape[1]] = blk
    return X


def allowed_pairs(pb):
    """Index arrays (a, b) of the two-site basis states with q_a + q_b = target,
    block after block, a major inside a block (the order of `psi_to_vec`)."""
    offA, _ = sector_offsets(pb.sectors_A)
    offB, _ = sector_offsets(pb.sectors_B)
    ia, ib = [], []
    for ai, bi in pb.psi_blocks():
        da, db = pb.sectors_A[ai][1], pb.sectors_B[bi][1]
        a = offA[ai] + np.arange(da)
        b = offB[bi] + np.arange(db)
        ia.append(np.repeat(a, db))
        ib.append(np.tile(b, da))
    return np.concatenate(ia), np.concatenate(ib)


def psi_to_vec(pb, psi=None):
    psi = pb.psi if psi is None else psi
    return np.concatenate([psi[k].reshape(-1) for k in pb.psi_blocks()])


def vec_to_psi(pb, x):
    out, o = {}, 0
    for ai, bi in pb.psi_blocks():
        da, db = pb.sectors_A[ai][1], pb.sectors_B[bi][1]
        out[(ai, bi)] = x[o:o + da * db].reshape(da, db)
        o += da * db
    return out


# ----------------------------------------------------------------------------
# T2: dense Kronecker assembly
# ----------------------------------------------------------------------------
def dense_heff(pb):
    """H_eff = Σ_k c_k kron(op_L P^π, op_R) restricted to the allowed (a,b) pairs.

    kron(X, Y)[(a′,b′),(a,b)] = X[a′,a]·Y[b′,b]; the restriction picks the rows
    and columns of the allowed pairs, so nothing else of the Kronecker product
    is ever formed (a 16384² dense matrix for config 1 would not fit)."""
    _, MA = sector_offsets(pb.sectors_A)
    _, MB = sector_offsets(pb.sectors_B)
    par = np.concatenate([np.full(d, 1.0 - 2.0 * sector_parity(q)) for q, d in pb.sectors_A])
    ia, ib = allowed_pairs(pb)
    H = np.zeros((len(ia), len(ia)))
    for k, (L, R, coef, tL, tR) in enumerate(pb.terms):
        X = np.eye(MA) if L is None else densify_op(pb.ops[L], pb.sectors_A, tL)
        Y = np.eye(MB) if R is None else densify_op(pb.ops[R], pb.sectors_B, tR)
        parity = 0
        if L is not None:
            parity = pb.ops[L]["parity"]
        elif R is not None:
            parity = pb.ops[R]["parity"]
        if parity:
            X = X * par[None, :]          # X · P : scales column a by (−1)^{N(q_a)}
        term = coef * X[np.ix_(ia, ia)] * Y[np.ix_(ib, ib)]
        if pb.block_coef is not None:     # the extra scalar belongs to the INPUT block: scale its columns
            o = 0
            for (ai, bi) in pb.psi_blocks():
                n = pb.sectors_A[ai][1] * pb.sectors_B[bi][1]
                term[:, o:o + n] *= pb.block_coef.get((k, (ai, bi)), 1.0)
                o += n
        H += term
    return H


def sigma_dense(pb, psi=None):
    """T2: σ = H_eff · vec(ψ), returned as blocks."""
    return vec_to_psi(pb, dense_heff(pb) @ psi_to_vec(pb, psi))


def full_kron_heff(pb):
    """The unrestricted Σ_k c_k kron(op_L P^π, op_R), (M_A·M_B)² — tiny inputs only."""
    _, MA = sector_offsets(pb.sectors_A)
    _, MB = sector_offsets(pb.sectors_B)
    par = np.concatenate([np.full(d, 1.0 - 2.0 * sector_parity(q)) for q, d in pb.sectors_A])
    H = np.zeros((MA * MB, MA * MB))
    for (L, R, coef, tL, tR) in pb.terms:
        X = np.eye(MA) if L is None else densify_op(pb.ops[L], pb.sectors_A, tL)
        Y = np.eye(MB) if R is None else densify_op(pb.ops[R], pb.sectors_B, tR)
        parity = pb.ops[L]["parity"] if L is not None else (pb.ops[R]["parity"] if R is not None else 0)
        if parity:
            X = X @ np.diag(par)
        H += coef * np.kron(X, Y)
    return H


# ----------------------------------------------------------------------------
# T3: block by block
# ----------------------------------------------------------------------------
def _applied_blocks(op, trans):
    """{col_sector: (row_sector, matrix)} of the operator as applied (after the
    optional transpose): maps input sector → (output sector, block)."""
    out = {}
    for (ri, ci), blk in op["blocks"].items():
        if trans:
            out[ri] = (ci, blk.T)
        else:
            out[ci] = (ri, blk)
    return out


def enumerate_tasks(pb):
    """All (k, input block, output block, Lblk, Rblk, coef·sign) triples."""
    blocks = set(pb.psi_blocks())
    tasks = []
    for k, (L, R, coef, tL, tR) in enumerate(pb.terms):
        La = None if L is None else _applied_blocks(pb.ops[L], tL)
        Ra = None if R is None else _applied_blocks(pb.ops[R], tR)
        parity = pb.ops[L]["parity"] if L is not None else (pb.ops[R]["parity"] if R is not None else 0)
        for (ai, bi) in pb.psi_blocks():
            if La is None:
                ao, Lb = ai, None
            elif ai in La:
                ao, Lb = La[ai]
            else:
                continue
            if Ra is None:
                bo, Rb = bi, None
            elif bi in Ra:
                bo, Rb = Ra[bi]
            else:
                continue
            if (ao, bo) not in blocks:
                continue
            sign = -1.0 if (parity and sector_parity(pb.sectors_A[ai][0])) else 1.0
            extra = 1.0 if pb.block_coef is None else pb.block_coef.get((k, (ai, bi)), 1.0)
            if extra == 0.0:
                continue
            tasks.append((k, (ai, bi), (ao, bo), Lb, Rb, coef * sign * extra))
    return tasks


def sigma_blockwise(pb, psi=None, naive=False):
    """T3: σ[a′,b′] += c_k·s · L_k[a′,a] ψ[a,b] R_k[b′,b]ᵀ over all tasks.

    ``naive=True`` replaces the two library products by explicit triple loops
    (tiny inputs; pins the use of the library routine)."""
    psi = pb.psi if psi is None else psi
    sigma = {k: np.zeros_like(v) for k, v in psi.items()}
    for (_, kin, kout, Lb, Rb, alpha) in enumerate_tasks(pb):
        x = psi[kin]
        if naive:
            t = x if Lb is None else _naive_matmul(Lb, x)
            y = t if Rb is None else _naive_matmul(t, Rb.T)
        else:
            t = x if Lb is None else Lb @ x
            y = t if Rb is None else t @ Rb.T
        sigma[kout] += alpha * y
    return sigma


def _naive_matmul(A, B):
    C = np.zeros((A.shape[0], B.shape[1]))
    for i in range(A.shape[0]):
        for j in range(B.shape[1]):
            s = 0.0
            for l in range(A.shape[1]):
                s += A[i, l] * B[l, j]
            C[i, j] = s
    return C


def flops_alg(pb):
    """Algorithmic flop count of one matvec:
    Σ_tasks min(2m′n(m+n′), 2mn′(n+m′)); an identity factor leaves one product."""
    total = 0
    for (_, (ai, bi), (ao, bo), Lb, Rb, _) in enumerate_tasks(pb):
        m, n = pb.sectors_A[ai][1], pb.sectors_B[bi][1]
        mo, no = pb.sectors_A[ao][1], pb.sectors_B[bo][1]
        if Lb is None and Rb is None:
            continue
        if Lb is None:
            total += 2 * m * n * no
        elif Rb is None:
            total += 2 * mo * m * n
        else:
            total += min(2 * mo * n * (m + no), 2 * m * no * (n + mo))
    return total


def diagonal_blockwise(pb):
    """diag(H_eff) as ψ-shaped blocks: only pairs whose applied L and R blocks are
    diagonal-sector (input sector = output sector) contribute,
    diag[a,b] = Σ_k c_k s · L_k[a,a] · R_k[b,b]."""
    out = {k: np.zeros((pb.sectors_A[k[0]][1], pb.sectors_B[k[1]][1])) for k in pb.psi_blocks()}
    for (_, kin, kout, Lb, Rb, alpha) in enumerate_tasks(pb):
        if kin != kout:
            continue
        dl = np.ones(out[kin].shape[0]) if Lb is None else np.diag(Lb)
        dr = np.ones(out[kin].shape[1]) if Rb is None else np.diag(Rb)
        out[kin] += alpha * np.outer(dl, dr)
    return out


def expectation_per_pair(pb, psi=None):
    """e_k = ⟨ψ, c_k (op_L(k) P^{π_k} ⊗ op_R(k)) ψ⟩ for every operator pair k, each from the blockwise
    definition applied to that pair alone (with the pair list {c†_i c_j} these are
    the elements γ_ij of the one-particle reduced density matrix)."""
    psi = pb.psi if psi is None else psi
    out = np.zeros(len(pb.terms))
    for k, term in enumerate(pb.terms):
        one = Problem(pb.n_charges, pb.sectors_A, pb.sectors_B, pb.target, pb.ops, [term], psi, pb.name)
        sig = sigma_blockwise(one)
        out[k] = sum(float(np.sum(sig[key] * psi[key])) for key in psi)
    return out
