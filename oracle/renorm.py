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


# ----------------------------------------------------------------------------
# Enlarging a block by a site (the other half of the renormalisation step)
# ----------------------------------------------------------------------------
# After the kept basis Φ has been applied, the next bond's enlarged block is A′ = (kept block) ⊗ (site).
# With the block's modes preceding the site's in the Jordan–Wigner string, a block operator x acts as
# x̃ ⊗ 1 and a site operator y as P^{π(y)} ⊗ ỹ, P = (−1)^{N_block}, so a product "block operator left of
# site operator" is (x̃ · P^π) ⊗ ỹ — the rule of SURVEY.md §8.0 with the site in the role of B.  Every
# operator the next bond needs on A′ is a sum of such products,
#
#       O_enl = Σ_j coef_j · (X_j · P^{π_j}) ⊗ y_j ,
#
# and by definition it equals Φ_{A′}† O Φ_{A′} with Φ_{A′} = Φ_kept ⊗ 1_site ("renormalized
# block operators"; PAPER.md:142 Ren_l / Ren_r).  `enlarge_dense` is the sum written out with explicit
# Kronecker products in the sector-major basis of A′; tests/test_oracle_enlarge.py pins it (and the
# product lists of the library's host builder) against the definition built from Fock-space matrices.
def enlarged_order(sectors_K, site_charges):
    """Sector-major ordering of the product basis |l⟩⊗|σ⟩ (l major): returns (perm, sectors_E) with
    perm[new index] = l·d + σ, charges ascending lexicographically, stable inside a sector — the
    ordering oracle.dmrg.sector_major gives kron_basis(left, site)."""
    qs = []
    for q, dim in sectors_K:
        qs += [tuple(q)] * dim
    d = len(site_charges)
    keys = [tuple(a + b for a, b in zip(ql, tuple(site_charges[s]))) for ql in qs for s in range(d)]
    perm = sorted(range(len(keys)), key=lambda i: (keys[i], i))
    sectors = []
    for i in perm:
        if sectors and sectors[-1][0] == keys[i]:
            sectors[-1][1] += 1
        else:
            sectors.append([keys[i], 1])
    return np.array(perm), [(k, n) for k, n in sectors]


def enlarge_dense(terms, sectors_K, site_charges):
    """Σ_j coef_j · kron(X_j P^{π_j}, y_j), rows and columns in the sector-major order of A′.

    terms: [(X dense M_K×M_K or None for the identity, y dense d×d, coef, π)], π = 1 if y is odd."""
    M = sum(dim for _, dim in sectors_K)
    d = len(site_charges)
    par = np.concatenate([np.full(dim, 1.0 - 2.0 * (int(sum(q)) % 2)) for q, dim in sectors_K]) if M else np.zeros(0)
    O = np.zeros((M * d, M * d))
    for X, y, coef, pi in terms:
        Xd = np.eye(M) if X is None else np.asarray(X, dtype=np.float64)
        if pi:
            Xd = Xd * par[None, :]
        O += coef * np.kron(Xd, np.asarray(y, dtype=np.float64))
    perm, _ = enlarged_order(sectors_K, site_charges)
    return O[np.ix_(perm, perm)]


def enlarged_order_right(sectors_K, site_charges):
    """As `enlarged_order` for the RIGHT block, product basis |σ⟩⊗|r⟩ with σ major: perm[new] = σ·M + r."""
    qs = []
    for q, dim in sectors_K:
        qs += [tuple(q)] * dim
    keys = [tuple(a + b for a, b in zip(tuple(site_charges[s]), qr)) for s in range(len(site_charges)) for qr in qs]
    perm = sorted(range(len(keys)), key=lambda i: (keys[i], i))
    sectors = []
    for i in perm:
        if sectors and sectors[-1][0] == keys[i]:
            sectors[-1][1] += 1
        else:
            sectors.append([keys[i], 1])
    return np.array(perm), [(k, n) for k, n in sectors]


def enlarge_dense_right(terms, sectors_K, site_charges, site_parity):
    """Σ_j coef_j · kron(y_j · P_s^{π_j}, X_j) for the right block B′ = site ⊗ kept (the site's modes precede
    the block's, so the parity P_s = diag(site_parity) of the SITE multiplies y when the block operator
    X_j is odd, π_j = 1), rows and columns in the sector-major order of B′.

    terms: [(X dense or None for the identity, y dense d×d, coef, π)]."""
    M = sum(dim for _, dim in sectors_K)
    d = len(site_charges)
    O = np.zeros((M * d, M * d))
    for X, y, coef, pi in terms:
        Xd = np.eye(M) if X is None else np.asarray(X, dtype=np.float64)
        yd = np.asarray(y, dtype=np.float64)
        if pi:
            yd = yd * np.asarray(site_parity, dtype=np.float64)[None, :]
        O += coef * np.kron(yd, Xd)
    perm, _ = enlarged_order_right(sectors_K, site_charges)
    return O[np.ix_(perm, perm)]
