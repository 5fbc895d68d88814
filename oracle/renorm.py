"""Renormalisation of block operators, O′ = Φ† O Φ (§II.A: "the renormalization step …
5–10 % of the run time"; Fig. 7 "Ren_l", "Ren_r").

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  After the two-site problem of a bond is solved,
the kept states of the enlarged block A = (left block ⊗ site) are the columns of an isometry
Φ (M_enl × M_new), block diagonal in the charge sectors (Φ[q]: dim_enl(q) × dim_new(q); a sector
whose states are all discarded has no block).  Every operator that the next bond needs is carried
into the new basis by the plain definition

    O′ = Φᵀ O Φ ,      per block   O′[q+δ, q] = Φ[q+δ]ᵀ · O[q+δ, q] · Φ[q] ,

real arithmetic, fp64.  `renormalise_dense` is that definition on densified matrices;
`renormalise_blockwise` is the same sum block by block (one dense product pair per block) and is what
large sizes use.  Pins: tests/test_oracle_renorm.py (brute-force element formula, identity and
orthogonal Φ, product homomorphism, and — the physics pin — the exported L_k of a DMRG bond carried
by the SVD basis of that bond equal Φ_new† X_k Φ_new built directly from the Fock-space matrices).
The paper prints no renormalised operator: "parity unpinned by the paper; pinned by definition".
"""
import numpy as np

from .heff import densify_op, sector_offsets


def densify_phi(phi, sectors_enl, sectors_new):
    """Dense M_enl × M_new matrix of Φ = {(enl sector index, new sector index): block}."""
    off_e, Me = sector_offsets(sectors_enl)
    off_n, Mn = sector_offsets(sectors_new)
    P = np.zeros((Me, Mn))
    for (ei, ni), blk in phi.items():
        P[off_e[ei]:off_e[ei] + blk.shape[0], off_n[ni]:off_n[ni] + blk.shape[1]] = blk
    return P


def renormalise_dense(op, sectors_enl, phi, sectors_new):
    """Φᵀ O Φ as a dense M_new × M_new matrix (the definition)."""
    P = densify_phi(phi, sectors_enl, sectors_new)
    return P.T @ densify_op(op, sectors_enl) @ P


def renormalise_blockwise(op, sectors_enl, phi, sectors_new):
    """{(row new-sector index, col new-sector index): Φ[q+δ]ᵀ O[q+δ,q] Φ[q]} for every stored block of
    ``op`` whose row and column sectors both survive in the new basis."""
    by_enl = {ei: (ni, blk) for (ei, ni), blk in phi.items()}
    out = {}
    for (ri, ci), blk in op["blocks"].items():
        if ri not in by_enl or ci not in by_enl:
            continue
        rn, Pr = by_enl[ri]
        cn, Pc = by_enl[ci]
        if Pr.shape[1] == 0 or Pc.shape[1] == 0:
            continue
        out[(rn, cn)] = Pr.T @ (blk @ Pc)
    return out


def flops(op, phi):
    """2·e′·e·n + 2·n′·e′·n per block (O Φ first, then Φᵀ ·): the count the library reports."""
    by_enl = {ei: blk.shape for (ei, ni), blk in phi.items()}
    total = 0
    for (ri, ci), blk in op["blocks"].items():
        if ri in by_enl and ci in by_enl and by_enl[ri][1] and by_enl[ci][1]:
            e_r, e_c = blk.shape
            n_r, n_c = by_enl[ri][1], by_enl[ci][1]
            total += 2 * e_r * e_c * n_c + 2 * n_r * e_r * n_c
    return total
