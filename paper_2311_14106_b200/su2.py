"""SU(2) spin-adapted H_eff for a spin-singlet target: host bookkeeping on top of the per-block-pair scalar of
`dmrgk_heff_create_blockcoef` ("the DMRG matrix and tensor algebra is
reformulated according to non-Abelian quantum numbers, thus the bond dimension D stands for the number of
renormalized multiplets"; BASELINE.json north_star: "SU(2) recoupling folded into per-block-pair scalar
coefficients").  No arithmetic of the matvec happens here: the GEMM kernels run the products, this module only
produces the scalar table they multiply in.

Conventions (the ones a spin-adapted DMRG hands over, stated so that the stored blocks are unambiguous):

* A sector of the left half is labelled (N, 2S), one of the right half (N, −2S): for total spin 0 the two halves
  of a ψ block carry the same S, so the two labels add up to the target (N_target, 0) and the U(1) block
  machinery of the library (sector index, ψ layout, task list) applies unchanged.  Sector dimensions count
  MULTIPLETS.  N + 2S is even for every sector, so the library's own fermionic sign never fires; the
  Jordan–Wigner sign of an odd pair, (−1)^{N_A} of the input A sector, is part of the scalar.
* An operator pair is Σ_q (T^k_q P^π) ⊗ Ũ^k_q with T^k a standard spherical tensor of rank k on the left half and
  Ũ^k_q = (−1)^{k−q} U^k_{−q}, U^k standard on the right half — the scalar product of two rank-k tensors.
  The stored blocks are REDUCED matrix elements in the Wigner–Eckart convention
      ⟨α′S′M′|T^k_q|αSM⟩ = ⟨S M k q|S′M′⟩ · ⟨α′S′‖T^k‖αS⟩ ;
  a rank-k operator is stored as one `dmrgk_op` per Δ(2S) ∈ {−2k, …, 2k}, with charge shift (ΔN, Δ2S) on the left
  and (−ΔN, −Δ2S) on the right half.
* With these conventions the recoupling coefficient of a block pair for total spin 0 — a 6j symbol with one
  zero argument, times the normalisation of the two singlet couplings — collapses to
      X(S → S′) = √((2S′+1)/(2S+1)) ,
  and it vanishes unless (S, k, S′) satisfy the triangle rule (`singlet_recoupling`).

Not built: targets with S ≠ 0 (several right-half sectors per left-half sector; 9j symbols).
"""
import math
import numpy as np

from . import problem


def triangle(two_a, two_b, two_c):
    """|a − b| ≤ c ≤ a + b and a + b + c integer, all arguments doubled."""
    return abs(two_a - two_b) <= two_c <= two_a + two_b and (two_a + two_b + two_c) % 2 == 0


def singlet_recoupling(two_s_in, two_s_out, two_k):
    """Scalar of the block pair (S → S′) of a rank-k pair for a spin-singlet target (module docstring)."""
    if two_s_in < 0 or two_s_out < 0 or not triangle(two_s_in, two_k, two_s_out):
        return 0.0
    return math.sqrt((two_s_out + 1.0) / (two_s_in + 1.0))


def block_coef_table(sectors_A, psi_blocks_a, pairs):
    """[K × n_blocks] scalars for `dmrgk_heff_create_blockcoef`.

    sectors_A: [((N, 2S), multiplets)], psi_blocks_a: A-sector index of every ψ block in layout order,
    pairs: [(two_k, parity, d2S)] per operator pair — its tensor rank (doubled), 1 for a fermionic pair, and the
    Δ(2S) of the stored left operator (None for a pair with an identity factor or a scalar: Δ = 0, rank 0)."""
    table = np.zeros((len(pairs), len(psi_blocks_a)))
    for k, (two_k, parity, d2) in enumerate(pairs):
        for j, a in enumerate(psi_blocks_a):
            N, two_s = sectors_A[a][0]
            x = singlet_recoupling(two_s, two_s + (d2 or 0), two_k or 0)
            table[k, j] = -x if (parity and N % 2) else x
    return table


def singlet_problem(sectors_A, sectors_B, n_target, ops, pairs, device=0, ctx=None, **opts):
    """DeviceProblem of a spin-singlet H_eff given in reduced form.

    ops: [{"half", "dq": (ΔN, ±Δ2S), "parity", "blocks": {(row sector, col sector): reduced block}}];
    pairs: [(L index or None, R index or None, coefficient, two_k)].  The rank of a pair and the Δ(2S) of its
    left operator fix the recoupling scalar of every block pair; the table is handed to the library once, at
    plan creation."""
    dp = problem.DeviceProblem(2, sectors_A, sectors_B, (n_target, 0), device, ctx)
    dp.create_ops([(o["half"], o["dq"], o["parity"]) for o in ops])
    dp.alloc_resident()
    for i, o in enumerate(ops):
        # a reduced block that vanishes identically (a selection rule) may be left out by the caller
        r, c, rows, cols = dp.ops[i].blocks()[:4]
        full = {(int(r[j]), int(c[j])): o["blocks"].get((int(r[j]), int(c[j])), np.zeros((int(rows[j]), int(cols[j]))))
                for j in range(len(r))}
        if set(o["blocks"]) - set(full):
            raise ValueError(f"singlet_problem: operator {i} has blocks outside its charge shift {o['dq']}")
        dp.set_op_host(i, full)
    meta = []
    for (L, R, coef, two_k) in pairs:
        if L is None or R is None:
            meta.append((0, 0, 0))
        else:
            if ops[L]["dq"][1] != -ops[R]["dq"][1] or ops[L]["dq"][0] != -ops[R]["dq"][0]:
                raise ValueError("singlet_problem: the two operators of a pair must carry opposite shifts")
            meta.append((two_k, ops[L]["parity"], ops[L]["dq"][1]))
    psi_a = [int(a) for a in dp.table[0]]
    bc = block_coef_table(sectors_A, psi_a, meta)
    dp.build([(L, R, coef, False, False) for (L, R, coef, _) in pairs], block_coef=bc, **opts)
    return dp


def pair_meta(ops, terms, ranks):
    """[(two_k, parity, Δ2S of the APPLIED left operator)] for `block_coef_table`, from operator specs with `.dq`,
    `.parity` (or dicts), terms (L, R, coef, trans_L, trans_R) and the doubled rank of every pair.  A pair applied
    through the transpose flags (the h.c. partner of a stored pair) shifts 2S the other way."""
    get = lambda o, k: o[k] if isinstance(o, dict) else getattr(o, k)
    meta = []
    for (L, R, _, trans_L, _), two_k in zip(terms, ranks):
        if L is None or R is None:
            meta.append((0, 0, 0))
        else:
            d2 = get(ops[L], "dq")[1]
            meta.append((two_k, get(ops[L], "parity"), -d2 if trans_L else d2))
    return meta
