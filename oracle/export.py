"""T1x: export of a DMRG bond as the block lists the GPU library consumes
(SURVEY.md §8(c) tier T1x; BASELINE.json: "complementary operators built on the
host").

At bond (i, i+1) the enlarged-block bases are Φ_A = Φ_L[i] ⊗ 1_site and
Φ_B = 1_site ⊗ Φ_R[i+2] (sector-major columns).  For every pair k of
`terms.complementary_terms` the renormalised block operators are
    L_k = Φ_A† X_k Φ_A      R_k = Φ_B† Y_k Φ_B ,
cut into U(1) blocks by the sector labels of Φ; entries outside the blocks
(q+dq, q) must vanish, which is asserted.  Since Φ_A Φ_A† commutes with the
sector structure but is not the identity once D truncates, Σ_k c_k (L_k P^π)⊗R_k
equals P†HP exactly only because each X_k ⊗ Y_k is projected as a whole:
P†(X⊗Y)P = (Φ_A†XΦ_A) ⊗ (Φ_B†YΦ_B).
"""
import numpy as np

from . import terms as terms_mod
from .dmrg import sector_slices
from .heff import Problem, sector_parity


def _cut_blocks(M, sectors, dq, tol=1e-11):
    index = {q: i for i, (q, _) in enumerate(sectors)}
    sl = sector_slices(sectors)
    blocks = {}
    mask = np.zeros(M.shape, dtype=bool)
    for ci, (q, _) in enumerate(sectors):
        r = index.get(tuple(a + b for a, b in zip(q, dq)))
        if r is None:
            continue
        blocks[(r, ci)] = M[sl[r], sl[ci]].copy()
        mask[sl[r], sl[ci]] = True
    leak = np.abs(M[~mask]).max() if (~mask).any() else 0.0
    assert leak < tol, f"operator leaks out of its charge blocks: {leak}"
    return blocks


def export_bond(dmrg, space, use_transpose_pairs=True, identity_as_none=True, prune=True):
    """`Problem` (without ψ) for the two-site space ``space`` of ``dmrg``."""
    n_A = space.A.n_modes
    tms = terms_mod.complementary_terms(dmrg.T, dmrg.V, n_A, dmrg.mc, prune=prune)
    PhiA, PhiB = space.A.Phi, space.B.Phi
    pb = Problem(dmrg.mc.shape[1], list(space.sectors_A), list(space.sectors_B), tuple(space.target),
                 name="T1x")
    stored = {}      # (family, label) -> (L op index, R op index, X, Y)
    partner_of = {"F1h": "F1", "F2h": "F2", "F3h": "F3"}
    for t in tms:
        Xd = PhiA.T @ (t.X @ PhiA)
        Yd = PhiB.T @ (t.Y @ PhiB)
        neg = tuple(-x for x in t.dq_A)
        # h.c. partner re-using the stored blocks through the transpose flags
        if use_transpose_pairs:
            key = None
            if t.family in partner_of:
                key = (partner_of[t.family], t.label)
            elif t.family == "F4" and t.label[0] > t.label[1]:
                key = ("F4", (t.label[1], t.label[0]))
            if key in stored:
                Li, Ri, X0, Y0 = stored[key]
                if np.abs(Xd - X0.T).max() < 1e-13 and np.abs(Yd - Y0.T).max() < 1e-13:
                    pb.terms.append((Li, Ri, t.coef, True, True))
                    continue
        Li = Ri = None
        if not (identity_as_none and t.family == "F0" and t.label == ("B",)):
            pb.ops.append({"half": "A", "dq": tuple(t.dq_A), "parity": t.parity,
                           "blocks": _cut_blocks(Xd, space.sectors_A, t.dq_A)})
            Li = len(pb.ops) - 1
        if not (identity_as_none and t.family == "F0" and t.label == ("A",)):
            pb.ops.append({"half": "B", "dq": neg, "parity": t.parity,
                           "blocks": _cut_blocks(Yd, space.sectors_B, neg)})
            Ri = len(pb.ops) - 1
        stored[(t.family, t.label)] = (Li, Ri, Xd, Yd)
        pb.terms.append((Li, Ri, t.coef, False, False))
    return pb
