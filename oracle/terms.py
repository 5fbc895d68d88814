"""Complementary-operator regrouping of Eq. (1) across a cut A|B.

The paper says only that H_eff is "built from renormalized block operators"
(PAPER.md:60); BASELINE.json's north_star fixes the form: σ = Σ_k c_k (L_k ⊗ R_k) ψ
with "complementary operators built on the host".  This module writes that sum
out for the general two-body Hamiltonian of PAPER.md:58,

    H = Σ_pq t_pq c†_p c_q + Σ_pqrs V_pqrs c†_p c†_q c_r c_s
      = Σ_pq t_pq c†_p c_q + ¼ Σ_pqrs W_pqrs c†_p c†_q c_r c_s ,
    W_pqrs = V_pqrs − V_qprs − V_pqsr + V_qpsr   (antisymmetrised),

with modes 0..n_A−1 in A (the enlarged left block) and the rest in B.  Every
cross term is brought to the canonical order "A-operator left of B-operator";
each operator of A anticommutes with each operator of B, which produces the
signs below.  In the product basis |a⟩⊗|b⟩ (A's modes precede B's in the
Jordan-Wigner string) an operator string X on A is X̃ ⊗ 1 and a string Y on B is
P_A^{π(Y)} ⊗ Ỹ, P_A = (−1)^{N_A}, tildes = matrices in the half's own JW basis.
Hence  X·Y = (X̃ P_A^π) ⊗ Ỹ  with π = 1 for a fermionic (odd) pair.

Families (derivation in the comments of `complementary_terms`):
  F0   H_A ⊗ 1 , 1 ⊗ H_B                                             coef +1
  F1   p∈B:  S^A_p ⊗ c̃†_p ,  S^A_p = Σ_{q∈A} t_pq c_q + ½Σ_{qrs∈A} W_pqrs c†_q c_r c_s   coef −1 (odd)
  F1h  s∈B:  S̄^A_s ⊗ c̃_s ,  S̄^A_s = Σ_{q∈A} t_qs c†_q + ½Σ_{pqr∈A} W_pqrs c†_p c†_q c_r  coef +1 (odd)
  F2   p∈A:  c̃†_p ⊗ S^B_p ,  S^B_p = ½Σ_{qrs∈B} W_pqrs c†_q c_r c_s                      coef +1 (odd)
  F2h  s∈A:  c̃_s ⊗ S̄^B_s ,  S̄^B_s = ½Σ_{pqr∈B} W_pqrs c†_p c†_q c_r                     coef −1 (odd)
  F3   p<q∈A: c†_p c†_q ⊗ P^B_pq , P^B_pq = Σ_{r<s∈B} W_pqrs c_r c_s                       coef +1 (even)
  F3h  r<s∈A: c_s c_r ⊗ P̄^B_rs ,  P̄^B_rs = Σ_{p<q∈B} W_pqsr c†_p c†_q                    coef +1 (even)
  F4   p,s∈A: c†_p c_s ⊗ Q^B_ps , Q^B_ps = Σ_{q,r∈B} W_pqrs c†_q c_r                       coef +1 (even)
For a Hermitian H the "h" families are the Hermitian conjugates of the plain
ones (S̄ = S†, P̄ = P†), but nothing here assumes it.  A pair whose coefficient
slice of (t, W) is identically zero is dropped (structural test on the
coefficients only) — this is the paper's "MPO bond dimension is much lower" in
real space.
"""
from dataclasses import dataclass
import numpy as np
import scipy.sparse as sp

from . import fock


@dataclass
class Term:
    X: object          # sparse 2^{n_A} matrix, A's own JW basis
    Y: object          # sparse 2^{n_B} matrix, B's own JW basis
    coef: float
    parity: int        # 1 if X and Y are fermionic (odd)
    dq_A: tuple        # charge shift of X on A (that of Y on B is the negative)
    family: str
    label: tuple = ()


def antisymmetrise(V):
    return V - V.transpose(1, 0, 2, 3) - V.transpose(0, 1, 3, 2) + V.transpose(1, 0, 3, 2)


def parity_operator(n):
    """P = (−1)^N on an n-mode Fock space (diagonal, sparse)."""
    occ = fock.occupations(n)
    return sp.diags((1 - 2 * (occ.sum(axis=1) % 2)).astype(np.float64), format="csr")


def _zero(n):
    return sp.csr_matrix((2 ** n, 2 ** n))


def complementary_terms(T, V, n_A, mode_charges, prune=True):
    """List of `Term` with  H = Σ_k coef_k · kron(X_k · P_A^{parity_k}, Y_k)."""
    n = T.shape[0]
    n_B = n - n_A
    mc = np.asarray(mode_charges, dtype=np.int64).reshape(n, -1)
    W = antisymmetrise(V)
    A = list(range(n_A))
    B = list(range(n_A, n))
    a = fock.annihilators(n_A)                      # a[p], p in A
    b = fock.annihilators(n_B)                      # b[p - n_A], p in B
    ad = [m.T.tocsr() for m in a]
    bd = [m.T.tocsr() for m in b]
    zero_q = tuple(0 for _ in range(mc.shape[1]))
    q = lambda p: tuple(int(x) for x in mc[p])
    neg = lambda t: tuple(-x for x in t)
    add = lambda s, t: tuple(x + y for x, y in zip(s, t))
    sA, sB = slice(0, n_A), slice(n_A, n)
    terms = []

    # F0 — all four (or both) indices in the same half: the half's own Eq. (1).
    H_A = fock.hamiltonian(T[sA, sA], V[sA, sA, sA, sA], a)
    H_B = fock.hamiltonian(T[sB, sB], V[sB, sB, sB, sB], b)
    terms.append(Term(H_A, sp.identity(2 ** n_B, format="csr"), 1.0, 0, zero_q, "F0", ("A",)))
    terms.append(Term(sp.identity(2 ** n_A, format="csr"), H_B, 1.0, 0, zero_q, "F0", ("B",)))

    # F1 — one creator in B, everything else in A.
    #   one-body: t_pq c†_p c_q (p∈B,q∈A) = −t_pq c_q c†_p
    #   two-body: the creator in B is p or q (equal by antisymmetry): 2·¼ = ½;
    #   c†_p (c†_q c_r c_s) = (−1)³ (c†_q c_r c_s) c†_p
    #   ⇒ −[Σ_q t_pq c_q + ½ Σ_qrs W_pqrs c†_q c_r c_s] · c†_p
    for p in B:
        if prune and not (np.any(T[p, sA]) or np.any(W[p, sA, sA, sA])):
            continue
        S = _zero(n_A)
        for qq in A:
            if T[p, qq] != 0.0:
                S = S + T[p, qq] * a[qq]
            for r in A:
                for s in A:
                    if W[p, qq, r, s] != 0.0:
                        S = S + 0.5 * W[p, qq, r, s] * (ad[qq] @ a[r] @ a[s])
        terms.append(Term(S.tocsr(), bd[p - n_A], -1.0, 1, neg(q(p)), "F1", (p,)))
    # F1h — one annihilator in B, everything else in A; already A-left:
    #   t_qs c†_q c_s (q∈A,s∈B) and ½ Σ_pqr W_pqrs (c†_p c†_q c_r) c_s
    for s in B:
        if prune and not (np.any(T[sA, s]) or np.any(W[sA, sA, sA, s])):
            continue
        S = _zero(n_A)
        for qq in A:
            if T[qq, s] != 0.0:
                S = S + T[qq, s] * ad[qq]
            for p in A:
                for r in A:
                    if W[p, qq, r, s] != 0.0:
                        S = S + 0.5 * W[p, qq, r, s] * (ad[p] @ ad[qq] @ a[r])
        terms.append(Term(S.tocsr(), b[s - n_A], +1.0, 1, q(s), "F1h", (s,)))
    # F2 — one creator in A, three operators in B; already A-left; the A–B
    #   hopping is entirely in F1/F1h, so there is no one-body part here.
    #   ½ Σ_qrs W_pqrs c†_p (c†_q c_r c_s)
    for p in A:
        if prune and not np.any(W[p, sB, sB, sB]):
            continue
        S = _zero(n_B)
        for qq in B:
            for r in B:
                for s in B:
                    if W[p, qq, r, s] != 0.0:
                        S = S + 0.5 * W[p, qq, r, s] * (bd[qq - n_A] @ b[r - n_A] @ b[s - n_A])
        terms.append(Term(ad[p], S.tocsr(), +1.0, 1, q(p), "F2", (p,)))
    # F2h — one annihilator in A, three operators in B:
    #   ½ Σ_pqr W_pqrs (c†_p c†_q c_r) c_s = (−1)³ ½ Σ W_pqrs c_s (c†_p c†_q c_r)
    for s in A:
        if prune and not np.any(W[sB, sB, sB, s]):
            continue
        S = _zero(n_B)
        for p in B:
            for qq in B:
                for r in B:
                    if W[p, qq, r, s] != 0.0:
                        S = S + 0.5 * W[p, qq, r, s] * (bd[p - n_A] @ bd[qq - n_A] @ b[r - n_A])
        terms.append(Term(a[s], S.tocsr(), -1.0, 1, neg(q(s)), "F2h", (s,)))
    # F3 — both creators in A, both annihilators in B:
    #   ¼ Σ_{pq∈A, rs∈B} = Σ_{p<q} Σ_{r<s} W_pqrs (c†_p c†_q)(c_r c_s)
    for p in A:
        for qq in A:
            if qq <= p:
                continue
            if prune and not np.any(W[p, qq, sB, sB]):
                continue
            P = _zero(n_B)
            for r in B:
                for s in B:
                    if r < s and W[p, qq, r, s] != 0.0:
                        P = P + W[p, qq, r, s] * (b[r - n_A] @ b[s - n_A])
            terms.append(Term(ad[p] @ ad[qq], P.tocsr(), +1.0, 0, add(q(p), q(qq)), "F3", (p, qq)))
    # F3h — both creators in B, both annihilators in A:
    #   Σ_{p<q∈B} Σ_{r<s∈A} W_pqrs c†_p c†_q c_r c_s ; the A pair is even and moves
    #   left freely; c_r c_s = −c_s c_r and −W_pqrs = W_pqsr
    #   ⇒ Σ_{r<s} (c_s c_r) · Σ_{p<q} W_pqsr c†_p c†_q
    for r in A:
        for s in A:
            if s <= r:
                continue
            if prune and not np.any(W[sB, sB, s, r]):
                continue
            P = _zero(n_B)
            for p in B:
                for qq in B:
                    if p < qq and W[p, qq, s, r] != 0.0:
                        P = P + W[p, qq, s, r] * (bd[p - n_A] @ bd[qq - n_A])
            terms.append(Term(a[s] @ a[r], P.tocsr(), +1.0, 0, neg(add(q(r), q(s))), "F3h", (r, s)))
    # F4 — one creator and one annihilator in each half: the four index patterns
    #   are equal by antisymmetry (4·¼ = 1):
    #   Σ W_pqrs c†_p c†_q c_r c_s (p,s∈A; q,r∈B) = Σ (c†_p c_s)(c†_q c_r)
    #   because the even B pair commutes with c_s.
    for p in A:
        for s in A:
            if prune and not np.any(W[p, sB, sB, s]):
                continue
            Q = _zero(n_B)
            for qq in B:
                for r in B:
                    if W[p, qq, r, s] != 0.0:
                        Q = Q + W[p, qq, r, s] * (bd[qq - n_A] @ b[r - n_A])
            terms.append(Term(ad[p] @ a[s], Q.tocsr(), +1.0, 0, add(q(p), neg(q(s))), "F4", (p, s)))
    return terms


def assemble(terms, n_A, n_B):
    """Σ_k coef_k · kron(X_k P_A^{π_k}, Y_k) as a sparse 2^{n_A+n_B} matrix."""
    P = parity_operator(n_A)
    H = sp.csr_matrix((2 ** (n_A + n_B), 2 ** (n_A + n_B)))
    for t in terms:
        XA = (t.X @ P) if t.parity else t.X
        H = H + t.coef * sp.kron(XA, t.Y, format="csr")
    return H
