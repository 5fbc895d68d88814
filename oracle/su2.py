"""ORACLE (test infrastructure, never imported by the product path): the SU(2) spin-adapted effective
Hamiltonian for a spin-singlet target.

PAPER.md:170-180 (§IV): "the SU(2) spin symmetry can also be utilized … the DMRG matrix and tensor algebra is
reformulated according to non-Abelian quantum numbers, thus the bond dimension D stands for the number of
renormalized multiplets"; BASELINE.json north_star: "SU(2) recoupling folded into per-block-pair scalar
coefficients".  The paper gives no formula (its algebra is in ref. [40]); what the adapted form must EQUAL has
a plain definition, and that definition is the oracle:

    H_red = Cᵀ H C ,   C = the isometry from the singlet-coupled multiplet basis
    |(α S_A, β S_B = S_A) 0 0⟩ = Σ_M ⟨S M S −M|0 0⟩ |α S M⟩|β S −M⟩      (`singlet_isometry`)

into the product space of the two halves, H the Fock-space Hamiltonian of Eq. (1).  Next to it
this module writes out, step by step, the adapted METHOD whose result must equal that definition
(`reduced_problem`):

  1. multiplet bases |α S M⟩ of each half with Condon–Shortley phases: highest-weight states = null space of
     S⁺ inside (N, S_z = S), the other M by S⁻ (`multiplets`);
  2. the cross-cut operator pairs of the complementary-operator regrouping (oracle/terms.py) recombined into
     pairs of STANDARD spherical tensor operators, H_cross = Σ_g Σ_q (T^k_q P^π) ⊗ Ũ^k_q with
     Ũ^k_q = (−1)^{k−q} U^k_{−q} (`tensor_groups`; standard means [S^z, T_q] = q T_q,
     [S^±, T_q] = √(k(k+1) − q(q±1)) T_{q±1}, checked by `tensor_defect`);
  3. reduced matrix elements by the Wigner–Eckart theorem in the convention
     ⟨α′S′M′|T^k_q|αSM⟩ = ⟨S M k q|S′M′⟩ · ⟨α′S′‖T^k‖αS⟩ (`reduce_tensor`);
  4. the recoupling scalar of a block pair for total spin 0, by brute-force summation of Clebsch–Gordan
     coefficients (`recoupling_singlet`), times the Jordan–Wigner sign (−1)^{π N_A};
  5. σ_red[a′,b′] += scalar · L_red[a′,a] ψ_red[a,b] R_red[b′,b]ᵀ — the block list of oracle/heff.py with
     `block_coef`, sectors labelled (N, 2S) on A and (N, −2S) on B so that charges add up to (N_target, 0); a
     rank-k operator is stored as one operator per Δ(2S) ∈ {−2k, …, 2k}.

All angular momenta are passed DOUBLED (integers 2j, 2m).  Not built: non-singlet targets (several B sectors
per A sector, 9j symbols) — "parity unpinned" does not apply: every function here is pinned in
tests/test_oracle_su2.py (CG against angular-momentum matrices and textbook values, tensors by their
commutators, Wigner–Eckart consistency over all M, method = definition, energies = exact diagonalisation).
"""
from dataclasses import dataclass, field
from math import factorial, sqrt
import numpy as np
import scipy.linalg
import scipy.sparse as sp

from . import fock, terms as oterms
from .heff import Problem


# ---------------------------------------------------------------------------------------------
# Clebsch–Gordan coefficients (Racah's closed form; Condon–Shortley phases)
# ---------------------------------------------------------------------------------------------
def cg(j1, m1, j2, m2, J, M):
    """⟨j1 m1 j2 m2 | J M⟩ with every argument doubled (integers)."""
    if m1 + m2 != M or abs(m1) > j1 or abs(m2) > j2 or abs(M) > J:
        return 0.0
    if (j1 + m1) % 2 or (j2 + m2) % 2 or (J + M) % 2 or (j1 + j2 + J) % 2:
        return 0.0
    if J > j1 + j2 or J < abs(j1 - j2):
        return 0.0
    h = lambda x: x // 2          # all arguments below are even
    f = factorial
    pref = (J + 1) * f(h(J + j1 - j2)) * f(h(J - j1 + j2)) * f(h(j1 + j2 - J)) / f(h(j1 + j2 + J) + 1)
    pref *= f(h(J + M)) * f(h(J - M)) * f(h(j1 - m1)) * f(h(j1 + m1)) * f(h(j2 - m2)) * f(h(j2 + m2))
    s = 0.0
    for k in range(0, h(j1 + j2 - J) + 1):
        a = [k, h(j1 + j2 - J) - k, h(j1 - m1) - k, h(j2 + m2) - k, h(J - j2 + m1) + k, h(J - j1 - m2) + k]
        if min(a) < 0:
            continue
        d = 1
        for x in a:
            d *= f(x)
        s += (-1) ** k / d
    return sqrt(pref) * s


# ---------------------------------------------------------------------------------------------
# spin operators and multiplet bases of a block of sites (modes (site↑, site↓), reading r8)
# ---------------------------------------------------------------------------------------------
def spin_operators(n_sites):
    """(S⁺, S⁻, S^z, N) on the 4^n_sites Fock space of a block, the block's own Jordan–Wigner basis."""
    a = fock.annihilators(2 * n_sites)
    dim = 2 ** (2 * n_sites)
    Sp = sp.csr_matrix((dim, dim))
    Sz = sp.csr_matrix((dim, dim))
    Nop = sp.csr_matrix((dim, dim))
    for s in range(n_sites):
        up, dn = a[2 * s], a[2 * s + 1]
        Sp = Sp + up.T @ dn
        Sz = Sz + 0.5 * (up.T @ up - dn.T @ dn)
        Nop = Nop + up.T @ up + dn.T @ dn
    return Sp.tocsr(), Sp.T.tocsr(), Sz.tocsr(), Nop.tocsr()


def multiplets(n_sites, keep=None, seed=None):
    """{(N, 2S): V} with V[:, α, i] = |α S M = S − i⟩ (Fock-space column vectors), i = 0 … 2S.

    Highest-weight states: an orthonormal basis of the null space of S⁺ restricted to the states with
    (N, S_z = S); lower states |S M−1⟩ = S⁻|S M⟩ / √(S(S+1) − M(M−1)) (Condon–Shortley).  `keep`
    (a fraction in (0, 1]) truncates in MULTIPLET space: the multiplets of a sector are mixed by a seeded
    random orthogonal matrix and the first ceil(keep·n) are kept ("D = renormalized multiplets")."""
    occ = fock.occupations(2 * n_sites)
    nup, ndn = occ[:, 0::2].sum(axis=1), occ[:, 1::2].sum(axis=1)
    Sp, Sm, _, _ = spin_operators(n_sites)
    Spd, Smd = Sp.toarray(), Sm.toarray()
    rng = np.random.default_rng(seed)
    out = {}
    for N in range(2 * n_sites + 1):
        for twoS in range(N % 2, min(N, 2 * n_sites - N) + 1, 2):
            u, d = (N + twoS) // 2, (N - twoS) // 2
            hi = np.flatnonzero((nup == u) & (ndn == d))
            if hi.size == 0:
                continue
            up = np.flatnonzero((nup == u + 1) & (ndn == d - 1))
            if up.size:
                ns = scipy.linalg.null_space(Spd[np.ix_(up, hi)], rcond=1e-12)
            else:
                ns = np.eye(hi.size)
            if ns.shape[1] == 0:
                continue
            if keep is not None:
                q, _ = np.linalg.qr(rng.normal(size=(ns.shape[1], ns.shape[1])))
                ns = (ns @ q)[:, :max(1, int(np.ceil(keep * ns.shape[1])))]
            V = np.zeros((Spd.shape[0], ns.shape[1], twoS + 1))
            V[hi, :, 0] = ns
            for i in range(1, twoS + 1):
                M2 = twoS - 2 * (i - 1)                       # doubled M of the state being lowered
                norm = sqrt((twoS * (twoS + 2) - M2 * (M2 - 2)) / 4.0)
                V[:, :, i] = Smd @ V[:, :, i - 1] / norm
            out[(N, twoS)] = V
    return out


# ---------------------------------------------------------------------------------------------
# step 2: pairs of standard tensor operators across the cut
# ---------------------------------------------------------------------------------------------
@dataclass
class TensorPair:
    """Σ_q (T_q P_A^parity) ⊗ Ũ_q ; U_{−q} = (−1)^{k−q} Ũ_q is the standard tensor on B."""
    k2: int                      # doubled rank
    parity: int
    dN_A: int                    # particle-number shift of T on A (that of U on B is the negative)
    T: dict                      # doubled q → sparse matrix on A
    Ut: dict                     # doubled q → sparse matrix Ũ_q on B   (None for an identity factor)
    family: str
    label: tuple = ()
    ident: str = ""              # "A" / "B" when that factor is the identity (family F0)

    def U(self):
        return {-q: ((-1) ** ((self.k2 - q) // 2)) * m for q, m in self.Ut.items()}


_R2 = 1.0 / sqrt(2.0)
# rank-½ combinations of the two spin components (index 0 = ↑, 1 = ↓): {2q: [(coefficient, spin)]}
_HALF_CREATION = {+1: [(1.0, 0)], -1: [(1.0, 1)]}                    # (c†_↑, c†_↓) and everything that transforms like it
_HALF_ANNIHILATION = {+1: [(1.0, 1)], -1: [(-1.0, 0)]}               # c̃ = (c_↓, −c_↑)
# two spin-½ operators on sites s ≠ s′, spin pairs (σ, σ′): {(2k, 2q): [(coefficient, (σ, σ′))]}
_PAIR_CC = {(2, 2): [(1.0, (0, 0))], (2, -2): [(1.0, (1, 1))],       # c†_{sσ} c†_{s′σ′}: CG coupling of two creation tensors
            (2, 0): [(_R2, (0, 1)), (_R2, (1, 0))], (0, 0): [(_R2, (0, 1)), (-_R2, (1, 0))]}
_PAIR_AA = {(2, 2): [(1.0, (1, 1))], (2, -2): [(1.0, (0, 0))],       # c_{s′σ′} c_{sσ} = (c†_{sσ} c†_{s′σ′})†: T̄^k_q = (−1)^{k−q} (T^k_{−q})†
            (2, 0): [(-_R2, (0, 1)), (-_R2, (1, 0))], (0, 0): [(_R2, (0, 1)), (-_R2, (1, 0))]}
_PAIR_CA = {(2, 2): [(1.0, (0, 1))], (2, -2): [(-1.0, (1, 0))],      # c†_{sσ} c_{s′σ′}: creation tensor coupled with c̃
            (2, 0): [(-_R2, (0, 0)), (_R2, (1, 1))], (0, 0): [(-_R2, (0, 0)), (-_R2, (1, 1))]}


def tensor_groups(T, V, n_sites_A):
    """The operator pairs of `terms.complementary_terms` (all of them: prune=False) recombined into TensorPairs.

    The recombination of the components of a group is orthogonal (signed Clebsch–Gordan matrices), so
    Σ_j c_j X_j ⊗ Y_j = Σ_{kq} T^k_q ⊗ Ũ^k_q with T^k_q = Σ_j O_{j,kq} X_j and Ũ^k_q = Σ_j O_{j,kq} c_j Y_j.
    Nothing here assumes H to be SU(2) invariant: whether the Ũ side comes out as a standard tensor is what
    `tensor_defect` tests."""
    n = T.shape[0]
    n_A = 2 * n_sites_A
    mc = np.zeros((n, 1), dtype=np.int64) + 1
    tl = oterms.complementary_terms(T, V, n_A, mc, prune=False)
    site, spin = (lambda p: p // 2), (lambda p: p % 2)
    groups = []
    by = {}
    for t in tl:
        by.setdefault(t.family, []).append(t)
    for t in by["F0"]:
        if t.label == ("A",):
            groups.append(TensorPair(0, 0, 0, {0: t.X}, {0: None}, "F0", ("A",), ident="B"))
        else:
            groups.append(TensorPair(0, 0, 0, {0: None}, {0: t.Y}, "F0", ("B",), ident="A"))

    def combine(table, comp):
        out = {}
        for key, lst in table.items():
            acc = None
            for c, s in lst:
                if s not in comp:
                    continue
                acc = c * comp[s] if acc is None else acc + c * comp[s]
            if acc is not None:
                out[key] = acc.tocsr()
        return out

    # rank ½: one group per site of the single operator
    for fam, table, dN in (("F1", _HALF_ANNIHILATION, -1), ("F1h", _HALF_CREATION, +1),
                           ("F2", _HALF_CREATION, +1), ("F2h", _HALF_ANNIHILATION, -1)):
        sites = {}
        for t in by.get(fam, []):
            sites.setdefault(site(t.label[0]), {})[spin(t.label[0])] = t
        for s, comp in sorted(sites.items()):
            X = combine(table, {sg: t.X for sg, t in comp.items()})
            Y = combine(table, {sg: t.coef * t.Y for sg, t in comp.items()})
            groups.append(TensorPair(1, 1, dN, X, Y, fam, (s,)))
    # ranks 0 and 1: one group per (ordered) site pair of the two operators
    for fam, table, dN in (("F3", _PAIR_CC, +2), ("F3h", _PAIR_AA, -2), ("F4", _PAIR_CA, 0)):
        pairs = {}
        for t in by.get(fam, []):
            p, q = t.label
            pairs.setdefault((site(p), site(q)), {})[(spin(p), spin(q))] = t
        for (s1, s2), comp in sorted(pairs.items()):
            if fam in ("F3", "F3h") and s1 == s2:
                # both operators on one site: only (↑, ↓) exists (p < q); c†_↑ c†_↓ is a scalar (k = 0)
                t = comp[(0, 1)]
                groups.append(TensorPair(0, 0, dN, {0: t.X.tocsr()}, {0: (t.coef * t.Y).tocsr()}, fam, (s1, s2)))
                continue
            X = combine(table, {sg: t.X for sg, t in comp.items()})
            Y = combine(table, {sg: t.coef * t.Y for sg, t in comp.items()})
            for k2 in (0, 2):
                Xk = {q: m for (kk, q), m in X.items() if kk == k2}
                Yk = {q: m for (kk, q), m in Y.items() if kk == k2}
                groups.append(TensorPair(k2, 0, dN, Xk, Yk, fam, (s1, s2)))
    return groups


def assemble_groups(groups, n_sites_A, n_sites_B):
    """Σ_g Σ_q (T_q P^π) ⊗ Ũ_q as a sparse matrix on the product Fock space (must equal terms.assemble)."""
    P = oterms.parity_operator(2 * n_sites_A)
    dA, dB = 4 ** n_sites_A, 4 ** n_sites_B
    H = sp.csr_matrix((dA * dB, dA * dB))
    for g in groups:
        for q, Tq in g.T.items():
            XA = sp.identity(dA, format="csr") if Tq is None else (Tq @ P if g.parity else Tq)
            Y = sp.identity(dB, format="csr") if g.Ut[q] is None else g.Ut[q]
            H = H + sp.kron(XA, Y, format="csr")
    return H


def tensor_defect(comps, k2, n_sites):
    """max-norm violation of the standard-tensor commutation relations by the components {2q: matrix}."""
    Sp, Sm, Sz, _ = spin_operators(n_sites)
    zero = sp.csr_matrix(Sp.shape)
    get = lambda q: comps.get(q, zero)
    worst = 0.0
    comm = lambda A, B: A @ B - B @ A
    for q in range(-k2, k2 + 1, 2):
        Tq = get(q)
        d = comm(Sz, Tq) - (q / 2.0) * Tq
        worst = max(worst, abs(d).max() if d.nnz else 0.0)
        for S, dq in ((Sp, +2), (Sm, -2)):
            c = sqrt(max(0.0, (k2 * (k2 + 2) - q * (q + dq)) / 4.0))
            d = comm(S, Tq) - c * get(q + dq)
            worst = max(worst, abs(d).max() if d.nnz else 0.0)
    return worst


# ---------------------------------------------------------------------------------------------
# step 3: Wigner–Eckart reduction
# ---------------------------------------------------------------------------------------------
def reduce_tensor(comps, k2, mults):
    """Reduced matrix elements {((N′, 2S′), (N, 2S)): ⟨α′S′‖T^k‖αS⟩ [n′ × n]} of a standard tensor between the
    multiplets `mults`, and the largest deviation between the values obtained from different (M, q) — the
    Wigner–Eckart theorem says there is none — including elements that must vanish."""
    red, defect = {}, 0.0
    dense = {q: (m.toarray() if sp.issparse(m) else np.asarray(m)) for q, m in comps.items()}
    for (N, tS), Vin in mults.items():
        for (N2, tS2), Vout in mults.items():
            vals = []
            for i in range(tS + 1):
                M = tS - 2 * i
                for q, Tq in dense.items():
                    M2 = M + q
                    if abs(M2) > tS2:
                        continue
                    me = Vout[:, :, (tS2 - M2) // 2].T @ (Tq @ Vin[:, :, i])
                    c = cg(tS, M, k2, q, tS2, M2)
                    if abs(c) > 1e-12:
                        vals.append(me / c)
                    else:
                        defect = max(defect, np.abs(me).max(initial=0.0))
            if not vals:
                continue
            ref = vals[0]
            for v in vals[1:]:
                defect = max(defect, np.abs(v - ref).max(initial=0.0))
            if np.abs(ref).max(initial=0.0) > 1e-13:
                red[((N2, tS2), (N, tS))] = ref
    return red, defect


# ---------------------------------------------------------------------------------------------
# step 4: recoupling for a singlet target, by brute force
# ---------------------------------------------------------------------------------------------
def recoupling_singlet(twoS_in, twoS_out, k2):
    """⟨(S′ S′) 0 0| Σ_q T^k_q ⊗ Ũ^k_q |(S S) 0 0⟩ / (⟨S′‖T‖S⟩⟨S′‖U‖S⟩), Ũ_q = (−1)^{k−q} U_{−q}: the sum over M, q of
    ⟨S′M′ S′−M′|00⟩ ⟨S M S −M|00⟩ (−1)^{k−q} ⟨S M k q|S′M′⟩ ⟨S −M k −q|S′ −M′⟩ — what a 6j symbol abbreviates."""
    s = 0.0
    for M in range(-twoS_in, twoS_in + 1, 2):
        for q in range(-k2, k2 + 1, 2):
            M2 = M + q
            if abs(M2) > twoS_out:
                continue
            s += (cg(twoS_out, M2, twoS_out, -M2, 0, 0) * cg(twoS_in, M, twoS_in, -M, 0, 0) * (-1) ** ((k2 - q) // 2)
                  * cg(twoS_in, M, k2, q, twoS_out, M2) * cg(twoS_in, -M, k2, -q, twoS_out, -M2))
    return s


# ---------------------------------------------------------------------------------------------
# the definition: singlet isometry, and the assembled reduced problem
# ---------------------------------------------------------------------------------------------
def sector_lists(multA, multB, N_target):
    """Sector lists of the reduced problem: A labelled (N, 2S), B labelled (N, −2S) (sorted), dims = multiplets."""
    sa = [((N, tS), V.shape[1]) for (N, tS), V in sorted(multA.items())]
    sb = [((N, -tS), V.shape[1]) for (N, tS), V in sorted(multB.items(), key=lambda kv: (kv[0][0], -kv[0][1]))]
    return sa, sb


def singlet_isometry(multA, multB, N_target):
    """C [dim_A·dim_B × n_red]: columns |(α S, β S) 0 0⟩ for every A sector (N_A, 2S) that has a partner
    (N_target − N_A, 2S) on B, in A-sector order, α-major, β-minor (the ψ-block order of oracle/heff.py)."""
    cols = []
    for (N, tS), VA in sorted(multA.items()):
        VB = multB.get((N_target - N, tS))
        if VB is None:
            continue
        for a in range(VA.shape[1]):
            for b in range(VB.shape[1]):
                v = 0.0
                for i in range(tS + 1):
                    M = tS - 2 * i
                    v = v + cg(tS, M, tS, -M, 0, 0) * np.kron(VA[:, a, i], VB[:, b, tS - i])
                cols.append(v)
    return np.array(cols).T


def reduced_problem(T, V, n_sites_A, N_target, keep=None, seed=0):
    """Steps 1-5: the spin-adapted block list (oracle.heff.Problem with block_coef) of the singlet sector with
    N_target particles, cut after `n_sites_A` sites.  Returns (Problem, multA, multB, groups, defects) where
    defects = {"tensor_A", "tensor_B", "wigner_eckart"} are the largest violations met on the way."""
    n_sites = T.shape[0] // 2
    n_sites_B = n_sites - n_sites_A
    multA = multiplets(n_sites_A, keep, seed)
    multB = multiplets(n_sites_B, keep, None if seed is None else seed + 1)
    groups = tensor_groups(T, V, n_sites_A)
    sa, sb = sector_lists(multA, multB, N_target)
    ia = {q: i for i, (q, _) in enumerate(sa)}
    ib = {q: i for i, (q, _) in enumerate(sb)}
    ops, tlist, bcoef, ranks = [], [], {}, []
    defects = {"tensor_A": 0.0, "tensor_B": 0.0, "wigner_eckart": 0.0}
    psi_blocks = [(ia[(N, tS)], ib[(N_target - N, -tS)]) for (N, tS), _ in sa if (N_target - N, -tS) in ib]
    for g in groups:
        if g.ident == "B":      # H_A ⊗ 1
            defects["tensor_A"] = max(defects["tensor_A"], tensor_defect(g.T, 0, n_sites_A))
            red, d = reduce_tensor(g.T, 0, multA)
            defects["wigner_eckart"] = max(defects["wigner_eckart"], d)
            ops.append({"half": "A", "dq": (0, 0), "parity": 0, "blocks": {(ia[o], ia[i]): m for (o, i), m in red.items()}})
            tlist.append((len(ops) - 1, None, 1.0, False, False))
            ranks.append(0)
            continue
        if g.ident == "A":      # 1 ⊗ H_B
            defects["tensor_B"] = max(defects["tensor_B"], tensor_defect(g.Ut, 0, n_sites_B))
            red, d = reduce_tensor(g.Ut, 0, multB)
            defects["wigner_eckart"] = max(defects["wigner_eckart"], d)
            ops.append({"half": "B", "dq": (0, 0), "parity": 0,
                        "blocks": {(ib[(o[0], -o[1])], ib[(i[0], -i[1])]): m for (o, i), m in red.items()}})
            tlist.append((None, len(ops) - 1, 1.0, False, False))
            ranks.append(0)
            continue
        U = g.U()
        defects["tensor_A"] = max(defects["tensor_A"], tensor_defect(g.T, g.k2, n_sites_A))
        defects["tensor_B"] = max(defects["tensor_B"], tensor_defect(U, g.k2, n_sites_B))
        redA, dA_ = reduce_tensor(g.T, g.k2, multA)
        redB, dB_ = reduce_tensor(U, g.k2, multB)
        defects["wigner_eckart"] = max(defects["wigner_eckart"], dA_, dB_)
        for d2 in range(-g.k2, g.k2 + 1, 2):      # one stored operator per Δ(2S)
            LA = {(ia[o], ia[i]): m for (o, i), m in redA.items() if o[1] - i[1] == d2 and o[0] - i[0] == g.dN_A}
            RB = {(ib[(o[0], -o[1])], ib[(i[0], -i[1])]): m for (o, i), m in redB.items()
                  if o[1] - i[1] == d2 and o[0] - i[0] == -g.dN_A}
            if not LA or not RB:
                continue
            ops.append({"half": "A", "dq": (g.dN_A, d2), "parity": g.parity, "blocks": LA})
            ops.append({"half": "B", "dq": (-g.dN_A, -d2), "parity": g.parity, "blocks": RB})
            k = len(tlist)
            tlist.append((len(ops) - 2, len(ops) - 1, 1.0, False, False))
            ranks.append(g.k2)
            for (a_idx, b_idx) in psi_blocks:
                N, tS = sa[a_idx][0]
                tS2 = tS + d2
                if tS2 < 0:
                    bcoef[(k, (a_idx, b_idx))] = 0.0
                    continue
                sign = -1.0 if (g.parity and N % 2) else 1.0       # Jordan–Wigner string of the B operator over A
                bcoef[(k, (a_idx, b_idx))] = sign * recoupling_singlet(tS, tS2, g.k2)
    pb = Problem(2, sa, sb, (N_target, 0), ops, tlist, {}, f"su2_singlet_N{N_target}", bcoef)
    pb.ranks = ranks            # doubled tensor rank of every pair (an input of the library's host code)
    return pb, multA, multB, groups, defects
