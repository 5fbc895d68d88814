"""Host builder of the block-enlargement step ("renormalized block
operators", Fig. 7 "Ren_l"; BASELINE.json: "complementary operators built on the host").

After the two-site problem of bond (A | B) is solved and the operators of A have been carried into the
kept basis (dmrgk_renorm: O′ = Φᵀ O Φ), the next bond's enlarged left block is A′ = (kept A) ⊗ (site s),
and every operator the next H_eff needs on A′ is a sum of products "kept operator ⊗ site operator",

        O_{A′} = Σ_j coef_j · (X_j · P^{π_j}) ⊗ y_j        (dmrgk_enlarge evaluates the sums on the GPU),

P = (−1)^{N_A} on the kept index, π_j = 1 when the site factor y_j is fermionic (the Jordan–Wigner string
of the site's modes runs over A).  This module produces the lists {(X_j, y_j, coef_j, π_j)} from the
one- and two-body coefficients t, V of Eq. (1) for the operator set of the left block:

    ("H",)            H_{A′}
    ("S", p)          S^{A′}_p = Σ_{q∈A′} t_pq c_q + ½ Σ_{q,r,s∈A′} W_pqrs c†_q c_r c_s    for p right of A′
    ("c+", p)         c†_p                  p ∈ A′
    ("c+c+", p, q)    c†_p c†_q             p < q ∈ A′
    ("c+c", p, s)     c†_p c_s              p ≤ s ∈ A′        (s < p is the transpose)

W is the antisymmetrised interaction (W_pqrs = V_pqrs − V_qprs − V_pqsr + V_qpsr, Σ V c†c†cc = ¼ Σ W c†c†cc).
The accumulation of S^{A′}_p — the complementary operator the left block carries — is where the O(k³)
coefficient sums of the method live; H_{A′} picks up the block–site coupling through S^A_p ⊗ c̃†_p (+h.c.)
and the pair–pair terms.  t and V are taken real with H Hermitian (t = tᵀ, W_pqrs = W_srqp), so adjoints of
kept operators are their transposes.

How a list is derived: every target is a polynomial in ladder operators; each monomial is split into its
kept part and its site part (moving the site operators to the right costs (−1)^{#(site op left of a kept
op)}), the kept part is matched to a stored operator or its transpose, the site part is multiplied out
as a d×d matrix in the site's own Jordan–Wigner basis.  Kept parts with three operators are never
expanded: summed with their coefficients they are S^A_p, which is stored.

Host logic only: index bookkeeping and coefficient sums in NumPy; no arithmetic on operator blocks.
The RIGHT block (site ⊗ kept B), which carries the complementary operators S^B, P^B, Q^B and their
accumulation, is the second half of this module (enlarge_right_lists).
"""
import numpy as np


def antisymmetrise(V):
    return V - V.transpose(1, 0, 2, 3) - V.transpose(0, 1, 3, 2) + V.transpose(1, 0, 3, 2)


class Site:
    """The d = 2^m states of a site with m modes, |n_0 … n_{m−1}⟩ = (c†_0)^{n_0}…|vac⟩, state index =
    Σ n_j 2^{m−1−j} (first mode most significant; reading r8 of DESIGN.md), its charges and its ladder
    operators with the Jordan–Wigner signs among the site's own modes."""

    def __init__(self, modes, mode_charges):
        self.modes = list(modes)
        m = len(self.modes)
        self.d = 2 ** m
        mc = np.asarray(mode_charges, dtype=np.int64)
        occ = np.array([[(i >> (m - 1 - j)) & 1 for j in range(m)] for i in range(self.d)], dtype=np.int64)
        self.charges = occ @ mc[self.modes]                                   # (d, n_charges)
        self.lower = {}
        for j, p in enumerate(self.modes):
            a = np.zeros((self.d, self.d))
            for i in range(self.d):
                if occ[i, j]:
                    a[i & ~(1 << (m - 1 - j)), i] = -1.0 if occ[i, :j].sum() % 2 else 1.0
            self.lower[p] = a

    def matrix(self, ops):
        """Product of ladder operators [(kind, mode)], written left to right as in the formula."""
        y = np.eye(self.d)
        for kind, p in ops:
            y = y @ (self.lower[p].T if kind == "+" else self.lower[p])
        return y


def _kept_part(ops):
    """A kept part (creators before annihilators, ≤ 2 operators) as (key, transposed, factor) of a stored
    operator; key None = identity; factor 0 = the monomial vanishes."""
    if not ops:
        return None, False, 1.0
    if len(ops) == 1:
        (k, p), = ops
        return ("c+", p), k == "-", 1.0
    (k1, p), (k2, q) = ops
    if k1 == "+" and k2 == "+":
        if p == q:
            return None, False, 0.0
        return (("c+c+", p, q), False, 1.0) if p < q else (("c+c+", q, p), False, -1.0)
    if k1 == "-" and k2 == "-":                       # c_p c_q = (c†_q c†_p)ᵀ
        if p == q:
            return None, False, 0.0
        return (("c+c+", q, p), True, 1.0) if q < p else (("c+c+", p, q), True, -1.0)
    if k1 == "+" and k2 == "-":                       # c†_p c_q ; for q < p it is (c†_q c_p)ᵀ
        return (("c+c", p, q), False, 1.0) if p <= q else (("c+c", q, p), True, 1.0)
    raise ValueError("kept part not in normal order")


class _Accumulator:
    """Σ of monomials of one target operator, grouped by (kept operator, transposed, site parity)."""

    def __init__(self, site, in_site):
        self.site, self.in_site, self.groups = site, in_site, {}

    def add(self, coef, ops):
        if coef == 0.0:
            return
        kept, sops, swaps, n_site_seen = [], [], 0, 0
        for op in ops:
            if op[1] in self.in_site:
                sops.append(op)
                n_site_seen += 1
            else:
                kept.append(op)
                swaps += n_site_seen                  # this kept operator jumps left over the site operators before it
        key, trans, factor = _kept_part(kept)
        if factor == 0.0:
            return
        sign = -1.0 if swaps % 2 else 1.0
        g = (key, trans, len(sops) % 2)
        y = self.groups.get(g)
        if y is None:
            y = self.groups[g] = np.zeros((self.site.d, self.site.d))
        y += coef * sign * factor * self.site.matrix(sops)

    def add_product(self, key, trans, coef, sops):
        """coef · (stored operator `key`, maybe transposed) ⊗ (site string), taken as given."""
        g = (key, trans, len(sops) % 2)
        y = self.groups.get(g)
        if y is None:
            y = self.groups[g] = np.zeros((self.site.d, self.site.d))
        y += coef * self.site.matrix(sops)

    def terms(self):
        return [(key, trans, y, pi) for (key, trans, pi), y in self.groups.items() if np.any(y)]


def enlarged_sectors(sectors_K, site_charges):
    """Sector list [(charge, dim)] of kept ⊗ site, charges ascending; dim = Σ over the kept sectors k with
    q′ − q_k a site charge (the sector-major product space dmrgk_enlarge expects)."""
    dims = {}
    for q, dim in sectors_K:
        if dim <= 0:
            continue
        for sq in site_charges:
            key = tuple(int(a) + int(b) for a, b in zip(q, sq))
            dims[key] = dims.get(key, 0) + dim
    return [(k, dims[k]) for k in sorted(dims)]


def left_block_keys(A, right):
    """Keys of the operator set the left block A carries when the modes `right` lie to its right."""
    A = list(A)
    keys = [("H",)] + [("S", p) for p in right] + [("c+", p) for p in A]
    keys += [("c+c+", p, q) for i, p in enumerate(A) for q in A[i + 1:]]
    keys += [("c+c", p, s) for i, p in enumerate(A) for s in A[i:]]
    return keys


def operator_spec(key, mode_charges):
    """(charge shift, parity) of a stored operator."""
    mc = np.asarray(mode_charges, dtype=np.int64)
    zero = np.zeros(mc.shape[1], dtype=np.int64)
    kind = key[0]
    if kind == "H":
        return tuple(int(x) for x in zero), 0
    if kind == "S":
        return tuple(int(x) for x in -mc[key[1]]), 1
    if kind == "c+":
        return tuple(int(x) for x in mc[key[1]]), 1
    if kind == "c+c+":
        return tuple(int(x) for x in mc[key[1]] + mc[key[2]]), 0
    if kind == "c+c":
        return tuple(int(x) for x in mc[key[1]] - mc[key[2]]), 0
    raise KeyError(key)


def enlarge_left_lists(T, V, mode_charges, A, S, right):
    """Product lists of every operator of the left block A′ = A ∪ S (S = the site's modes, all to the
    right of A's), `right` = the modes to the right of A′.

    Returns (site, {target key: [(kept key or None, transposed, y (d×d), π)]}).  The kept keys refer to
    the operator set of A with S ∪ right to its right (left_block_keys(A, S + right))."""
    T = np.asarray(T, dtype=np.float64)
    W = antisymmetrise(np.asarray(V, dtype=np.float64))
    A, S, right = list(A), list(S), list(right)
    site = Site(S, mode_charges)
    in_site = set(S)
    Ap = A + S
    out = {}

    def acc():
        return _Accumulator(site, in_site)

    # bare operators: one monomial each
    for p in Ap:
        a = acc()
        a.add(1.0, [("+", p)])
        out[("c+", p)] = a.terms()
    for i, p in enumerate(Ap):
        for q in Ap[i + 1:]:
            a = acc()
            a.add(1.0, [("+", p), ("+", q)])
            out[("c+c+", p, q)] = a.terms()
        for s in Ap[i:]:
            a = acc()
            a.add(1.0, [("+", p), ("-", s)])
            out[("c+c", p, s)] = a.terms()

    # S^{A′}_p, p to the right of A′: the all-in-A part is the stored S^A_p; every other monomial has at
    # most two kept operators
    for p in right:
        a = acc()
        a.add_product(("S", p), False, 1.0, [])
        for q in S:
            a.add(T[p, q], [("-", q)])
        for q in Ap:
            for r in Ap:
                for s in Ap:
                    if q in in_site or r in in_site or s in in_site:
                        a.add(0.5 * W[p, q, r, s], [("+", q), ("-", r), ("-", s)])
        out[("S", p)] = a.terms()

    # H_{A′} = H_A ⊗ 1 + 1 ⊗ H_S + block–site coupling.  Monomials with exactly ONE site operator sum to
    # −(S^A_p P) ⊗ c̃†_p + ((S^A_p)ᵀ P) ⊗ c̃_p (p ∈ S): t_pq c†_p c_q = −c_q c†_p for p ∈ S, q ∈ A, and the
    # three-kept-operator strings carry (−1)³ likewise; all other cross monomials have ≤ 2 kept operators.
    a = acc()
    a.add_product(("H",), False, 1.0, [])
    for p in S:
        a.add_product(("S", p), False, -1.0, [("+", p)])
        a.add_product(("S", p), True, +1.0, [("-", p)])
    for p in S:
        for q in S:
            a.add(T[p, q], [("+", p), ("-", q)])
    for p in Ap:
        for q in Ap:
            for r in Ap:
                for s in Ap:
                    n_site = (p in in_site) + (q in in_site) + (r in in_site) + (s in in_site)
                    if n_site >= 2:
                        a.add(0.25 * W[p, q, r, s], [("+", p), ("+", q), ("-", r), ("-", s)])
    out[("H",)] = a.terms()
    return site, out


# ----------------------------------------------------------------------------
# RIGHT block: B′ = (site s) ⊗ (kept B), the site's modes precede B's in the Jordan–Wigner string
# ----------------------------------------------------------------------------
# The right block carries the COMPLEMENTARY operators of the regrouping: for the modes
# `left` to the left of the block
#     ("H",)           H_{B}
#     ("c+", p)        c†_p                                   p ∈ B
#     ("S", p)         S^B_p  = ½ Σ_{q,r,s∈B} W_pqrs c†_q c_r c_s          p ∈ left   (no one-body part)
#     ("P", p, q)      P^B_pq = Σ_{r<s∈B} W_pqrs c_r c_s                   p < q ∈ left
#     ("Q", p, s)      Q^B_ps = Σ_{q,r∈B} W_pqrs c†_q c_r                  p ≤ s ∈ left  (Q_sp = Q_psᵀ)
# With the site to the LEFT of the kept block a product "site operator left of block operator" is
# (y · P_s^{π_x}) ⊗ X: the parity now sits on the small site factor (P_s = (−1)^{n_σ}, π_x = parity of the
# block operator) and is folded into the d×d matrix on the host; the enlarged basis is ordered
# |σ⟩ ⊗ |r⟩ with σ major.  Accumulating S, P and Q here is where the sums over the interaction live:
#     P^{B′}_pq = P^B_pq + Σ_{(r,s) not both in B} ½ W_pqrs c_r c_s
#     Q^{B′}_ps = Q^B_ps + Σ_{(q,r) not both in B} W_pqrs c†_q c_r
#     S^{B′}_p  = S^B_p + Σ_{q∈s} c̃†_q ⊗ P^B_pq + Σ_{s∈s} c̃_s ⊗ Q^B_ps + (monomials with ≥ 2 site operators)
#     H_{B′}    = H_B + H_s + Σ_{p∈s} [c̃†_p P_s ⊗ S^B_p − c̃_p P_s ⊗ (S^B_p)ᵀ] + Σ_{p<q∈s} [c̃†_p c̃†_q ⊗ P^B_pq + c̃_q c̃_p ⊗ (P^B_pq)ᵀ]
#                 + Σ_{p,s∈s} c̃†_p c̃_s ⊗ Q^B_ps + (monomials with ≤ 1 block operator)
# (second line of S^{B′}: the r∈s and s∈s placements of ½ W c†_q c_r c_s are equal by W_pqrs = −W_pqsr.)
def right_block_keys(B, left):
    left = list(left)
    keys = [("H",)] + [("c+", p) for p in B] + [("S", p) for p in left]
    keys += [("P", p, q) for i, p in enumerate(left) for q in left[i + 1:]]
    keys += [("Q", p, s) for i, p in enumerate(left) for s in left[i:]]
    return keys


def right_operator_spec(key, mode_charges):
    mc = np.asarray(mode_charges, dtype=np.int64)
    kind = key[0]
    if kind in ("H", "c+"):
        return operator_spec(key, mode_charges)
    if kind == "S":                                   # pairs with c†_p on the left block: shift −q_p
        return tuple(int(x) for x in -mc[key[1]]), 1
    if kind == "P":
        return tuple(int(x) for x in -(mc[key[1]] + mc[key[2]])), 0
    if kind == "Q":
        return tuple(int(x) for x in -(mc[key[1]] - mc[key[2]])), 0
    raise KeyError(key)


def right_key_parity(key):
    """Fermion parity of a stored right-block operator (None = identity)."""
    return 1 if key is not None and key[0] in ("c+", "S") else 0


def fold_site_parity(site, key, y):
    """y · P_s^{π_x}: the form dmrgk_enlarge takes for the right block (site_major = 1)."""
    return y * site.parity[None, :] if right_key_parity(key) else y


class _RightAccumulator(_Accumulator):
    """Monomials whose block part has at most one operator; the site part stays on the left."""

    def add(self, coef, ops):
        if coef == 0.0:
            return
        kept, sops, swaps, n_kept_seen = [], [], 0, 0
        for op in ops:
            if op[1] in self.in_site:
                sops.append(op)
                swaps += n_kept_seen                  # this site operator jumps left over the block operators before it
            else:
                kept.append(op)
                n_kept_seen += 1
        if len(kept) > 1:
            raise ValueError("block part with more than one operator must be given as a stored sum")
        key, trans, factor = _kept_part(kept)
        sign = -1.0 if swaps % 2 else 1.0
        self.add_product(key, trans, coef * sign * factor, sops, len(kept) % 2)

    def add_product(self, key, trans, coef, sops, kept_parity):
        """coef · (site string · P_s^{kept parity}) ⊗ (stored operator `key`, maybe transposed)."""
        assert kept_parity == right_key_parity(key)
        y = self.site.matrix(sops)                    # P_s^{kept parity} is applied by the consumer (fold_site_parity)
        g = (key, trans, len(sops) % 2)
        acc = self.groups.get(g)
        if acc is None:
            acc = self.groups[g] = np.zeros((self.site.d, self.site.d))
        acc += coef * y


def enlarge_right_lists(T, V, mode_charges, left, S, B):
    """Product lists of every operator of the right block B′ = S ∪ B (S = the site's modes, all to the left
    of B's), `left` = the modes to the left of B′.  Kept keys refer to right_block_keys(B, left + S).

    Returns (site, {target key: [(kept key or None, transposed, y (d×d), site factor odd)]}); the product is
    (y · P_s^{π_x}) ⊗ X with π_x = right_key_parity(kept key) — see fold_site_parity."""
    T = np.asarray(T, dtype=np.float64)
    W = antisymmetrise(np.asarray(V, dtype=np.float64))
    left, S, B = list(left), list(S), list(B)
    site = Site(S, mode_charges)
    m = len(S)
    site.parity = np.array([1.0 - 2.0 * (bin(i).count("1") % 2) for i in range(site.d)])
    in_site, in_B = set(S), set(B)
    Bp = S + B
    out = {}

    def acc():
        return _RightAccumulator(site, in_site)

    for p in Bp:
        a = acc()
        a.add(1.0, [("+", p)])
        out[("c+", p)] = a.terms()
    for i, p in enumerate(left):
        # S^{B′}_p
        a = acc()
        a.add_product(("S", p), False, 1.0, [], 1)
        for q in S:
            a.add_product(("P", p, q), False, 1.0, [("+", q)], 0)
            a.add_product(("Q", p, q), False, 1.0, [("-", q)], 0)
        for q in Bp:
            for r in Bp:
                for s in Bp:
                    if (q in in_site) + (r in in_site) + (s in in_site) >= 2:
                        a.add(0.5 * W[p, q, r, s], [("+", q), ("-", r), ("-", s)])
        out[("S", p)] = a.terms()
        for q in left[i + 1:]:
            a = acc()
            a.add_product(("P", p, q), False, 1.0, [], 0)
            for r in Bp:
                for s in Bp:
                    if r in in_site or s in in_site:
                        a.add(0.5 * W[p, q, r, s], [("-", r), ("-", s)])
            out[("P", p, q)] = a.terms()
        for s in left[i:]:
            a = acc()
            a.add_product(("Q", p, s), False, 1.0, [], 0)
            for q in Bp:
                for r in Bp:
                    if q in in_site or r in in_site:
                        a.add(W[p, q, r, s], [("+", q), ("-", r)])
            out[("Q", p, s)] = a.terms()
    # H_{B′}
    a = acc()
    a.add_product(("H",), False, 1.0, [], 0)
    for p in S:
        a.add_product(("S", p), False, +1.0, [("+", p)], 1)
        a.add_product(("S", p), True, -1.0, [("-", p)], 1)
    for i, p in enumerate(S):
        for q in S[i + 1:]:
            a.add_product(("P", p, q), False, 1.0, [("+", p), ("+", q)], 0)
            a.add_product(("P", p, q), True, 1.0, [("-", q), ("-", p)], 0)
        for s in S:
            if p <= s:
                a.add_product(("Q", p, s), False, 1.0, [("+", p), ("-", s)], 0)
            else:
                a.add_product(("Q", s, p), True, 1.0, [("+", p), ("-", s)], 0)
    for p in Bp:
        for q in Bp:
            if p in in_site or q in in_site:
                a.add(T[p, q], [("+", p), ("-", q)])
    for p in Bp:
        for q in Bp:
            for r in Bp:
                for s in Bp:
                    if (p in in_site) + (q in in_site) + (r in in_site) + (s in in_site) >= 3:
                        a.add(0.25 * W[p, q, r, s], [("+", p), ("+", q), ("-", r), ("-", s)])
    out[("H",)] = a.terms()
    return site, out
