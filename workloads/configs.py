"""The BASELINE.json workloads as seeded *inputs* (structure + values).

A workload is: two sector lists (enlarged left block A, enlarged right block B),
a target charge, a list of stored operators (each a set of blocks (q+dq, q) on
one half with an RNG stream for its values) and a list of operator-pair terms
(L index, R index, coefficient, transpose flags).  What the terms *mean* — the
product, the fermionic sign, the accumulation — is the method and lives in
``oracle/`` and in the CUDA library, separately.

Sources: BASELINE.json configs; SURVEY.md §8.0 (term families F0-F4 and their
counts, which follow from PAPER.md Eq. (1), line 58), §8(c) readings r14-r18,
§8(d) concrete inputs.  The paper's own operator values (converged DMRG
environments in its optimised bases) are not available, so the *structure* is
the lattice's and the *values* are synthetic (r17).
"""
from dataclasses import dataclass, field
from itertools import product
import math
import numpy as np

from .rng import normal12, uniform_u64
from .sectors import gaussian_sectors, binom

PSI_STREAM = 7
COEF_STREAM = 9
SHIFT_STREAM = 11
OP_STREAM0 = 16


def op_stream_id(op_index):
    return OP_STREAM0 + op_index


def op_stream_of(wl, op_index):
    """RNG stream of stored operator ``op_index`` of ``wl`` (its own if pinned by sub_workload)."""
    s = wl.ops[op_index].stream
    return s if s >= 0 else op_stream_id(op_index)


@dataclass
class OpSpec:
    half: str            # "A" or "B"
    dq: tuple            # charge shift: blocks (row sector q+dq, column sector q)
    parity: int          # 0 even, 1 odd (fermionic)
    symmetric: bool = False   # dq == 0 and every diagonal block symmetrised
    scale_mode: str = "rsqrt_cols"   # "one" (config 2) or "rsqrt_cols" (configs 3-5)
    tag: str = ""
    stream: int = -1     # RNG stream of the values; −1 = op_stream_id(position in wl.ops).  Set when an
                         # operator keeps its values while moving to another position (sub_workload)


@dataclass
class TermSpec:
    L: object            # index into ops, or None for the identity on A
    R: object            # index into ops, or None for the identity on B
    coef: float
    trans_L: bool = False
    trans_R: bool = False
    family: str = ""


@dataclass
class Workload:
    name: str
    seed: int
    n_charges: int
    sectors_A: list      # [(charge tuple, dim)]
    sectors_B: list
    target: tuple
    ops: list = field(default_factory=list)
    terms: list = field(default_factory=list)
    hermitian: bool = False

    @property
    def M_A(self):
        return sum(d for _, d in self.sectors_A)

    @property
    def M_B(self):
        return sum(d for _, d in self.sectors_B)

    def sectors(self, half):
        return self.sectors_A if half == "A" else self.sectors_B


# ----------------------------------------------------------------------------
# block tables (pure index bookkeeping; the library recomputes its own)
# ----------------------------------------------------------------------------
def _add(q, dq):
    return tuple(a + b for a, b in zip(q, dq))


def op_block_table(sectors, dq):
    """Blocks of an operator with shift dq: [(row_idx, col_idx, rows, cols, offset)].

    One block for every column sector q (in sector order) such that q+dq is also
    a sector; offsets count *unpadded* elements, block after block.
    """
    index = {q: i for i, (q, _) in enumerate(sectors)}
    out, off = [], 0
    for ci, (q, cols) in enumerate(sectors):
        r = index.get(_add(q, dq))
        if r is None or cols == 0 or sectors[r][1] == 0:
            continue
        rows = sectors[r][1]
        out.append((r, ci, rows, cols, off))
        off += rows * cols
    return out


def psi_block_table(sectors_A, sectors_B, target):
    """ψ blocks (qA, qB) with qA+qB = target, in A-sector order."""
    index_B = {q: i for i, (q, _) in enumerate(sectors_B)}
    out, off = [], 0
    for ai, (qa, rows) in enumerate(sectors_A):
        qb = tuple(t - a for t, a in zip(target, qa))
        bi = index_B.get(qb)
        if bi is None or rows == 0 or sectors_B[bi][1] == 0:
            continue
        cols = sectors_B[bi][1]
        out.append((ai, bi, rows, cols, off))
        off += rows * cols
    return out


# ----------------------------------------------------------------------------
# values
# ----------------------------------------------------------------------------
def _block_scale(spec, cols):
    return 1.0 if spec.scale_mode == "one" else 1.0 / math.sqrt(cols)


def fill_op_host(wl, op_index, only_blocks=None):
    """Blocks of stored operator ``op_index`` as {(row_idx, col_idx): ndarray}.

    value(r, c) = scale * g(off + r*cols + c), g = normal12 of the operator's
    stream; for a ``symmetric`` operator a (square, diagonal-sector) block is
    0.5*(g(r,c) + g(c,r)) * scale.  ``only_blocks`` restricts to a set of
    (row_idx, col_idx) keys (used to regenerate sampled blocks at full size).
    """
    spec = wl.ops[op_index]
    sectors = wl.sectors(spec.half)
    stream = op_stream_of(wl, op_index)
    out = {}
    for (ri, ci, rows, cols, off) in op_block_table(sectors, spec.dq):
        if only_blocks is not None and (ri, ci) not in only_blocks:
            continue
        idx = off + np.arange(rows * cols, dtype=np.uint64).reshape(rows, cols)
        g = normal12(wl.seed, stream, idx)
        if spec.symmetric:
            assert ri == ci and rows == cols
            g = (g + g.T) * 0.5
        out[(ri, ci)] = g * _block_scale(spec, cols)
    return out


def fill_psi_host(wl, stream=PSI_STREAM):
    """ψ blocks {(a_idx, b_idx): ndarray} with N(0,1)-like entries (normal12)."""
    out = {}
    for (ai, bi, rows, cols, off) in psi_block_table(wl.sectors_A, wl.sectors_B, wl.target):
        idx = off + np.arange(rows * cols, dtype=np.uint64).reshape(rows, cols)
        out[(ai, bi)] = normal12(wl.seed, stream, idx)
    return out


# ----------------------------------------------------------------------------
# config 2: synthetic block-sparse matvec (BASELINE.json configs[1]; r14, r15)
# ----------------------------------------------------------------------------
def synthetic_config2(M=1024, n_q=33, K=512, seed=2, width2=32.0, name=None):
    """U(1) charge, sectors q=0..n_q-1 ∝ exp(-(q-c)²/width2) with c=(n_q-1)/2,
    ψ blocks where qA+qB = n_q-1, K pairs with δ_L uniform in {-2..2},
    δ_R = -δ_L, parity δ_L mod 2, entries and c_k N(0,1).  Not symmetric."""
    c = (n_q - 1) / 2.0
    w = [math.exp(-((q - c) ** 2) / width2) for q in range(n_q)]
    caps = [binom(n_q - 1, q) for q in range(n_q)]
    dims = gaussian_sectors(M, w, caps)
    sectors = [((q,), d) for q, d in enumerate(dims)]
    wl = Workload(name or f"config2_M{M}_K{K}", seed, 1, sectors, list(sectors), (n_q - 1,))
    shifts = (uniform_u64(seed, SHIFT_STREAM, np.arange(K)) % np.uint64(5)).astype(np.int64) - 2
    coefs = normal12(seed, COEF_STREAM, np.arange(K))
    for k in range(K):
        d = int(shifts[k])
        wl.ops.append(OpSpec("A", (d,), d & 1, False, "one", f"L{k}"))
        wl.ops.append(OpSpec("B", (-d,), d & 1, False, "one", f"R{k}"))
        wl.terms.append(TermSpec(2 * k, 2 * k + 1, float(coefs[k]), False, False, "syn"))
    return wl


# ----------------------------------------------------------------------------
# configs 3-5: lattice-shaped operator-pair lists (SURVEY §8.0 families)
# ----------------------------------------------------------------------------
def _family_builder(wl, mode_shifts_A, mode_shifts_B, pair_fraction=None, keep=None):
    """Append ops and terms of families F0-F4 for modes with the given charge
    shifts (one tuple per mode = the shift of its creation operator).

    Hermitian construction (r18): every δ≠0 (or p≠s) pair is stored once and its
    h.c. partner re-uses the same stored blocks through the transpose flags,
    with coefficient −c for fermionic (odd) pairs and +c for even ones; the
    self-adjoint operators (H_A, H_B, c†_p c_p and its complement) have
    symmetrised blocks.  ``keep(family, ordinal)`` may thin the list (used for
    scaled-down copies and for the executed subset of config 5).
    """
    zero = tuple(0 for _ in wl.target)
    neg = lambda d: tuple(-x for x in d)
    add = lambda a, b: tuple(x + y for x, y in zip(a, b))
    keep = keep or (lambda fam, i: True)

    def new_op(half, dq, parity, sym, tag):
        wl.ops.append(OpSpec(half, tuple(dq), parity, sym, "rsqrt_cols", tag))
        return len(wl.ops) - 1

    def pair(Lop, Rop, coef, fam, partner_coef=None):
        wl.terms.append(TermSpec(Lop, Rop, coef, False, False, fam))
        if partner_coef is not None:
            wl.terms.append(TermSpec(Lop, Rop, partner_coef, True, True, fam + "^hc"))

    # F0: H_A ⊗ 1 and 1 ⊗ H_B
    hA = new_op("A", zero, 0, True, "H_A")
    hB = new_op("B", zero, 0, True, "H_B")
    wl.terms.append(TermSpec(hA, None, 1.0, False, False, "F0"))
    wl.terms.append(TermSpec(None, hB, 1.0, False, False, "F0"))
    # F1: for p in B:  −S^A_p ⊗ c†_p  and  +S^A_p† ⊗ c_p
    for i, s in enumerate(mode_shifts_B):
        if not keep("F1", i):
            continue
        Lop = new_op("A", neg(s), 1, False, f"S^A_{i}")
        Rop = new_op("B", s, 1, False, f"c†_B{i}")
        pair(Lop, Rop, -1.0, "F1", +1.0)
    # F2: for p in A:  +c†_p ⊗ S^B_p  and  −c_p ⊗ S^B_p†
    cdag_A = {}
    for i, s in enumerate(mode_shifts_A):
        if not keep("F2", i):
            continue
        Lop = new_op("A", s, 1, False, f"c†_A{i}")
        Rop = new_op("B", neg(s), 1, False, f"S^B_{i}")
        cdag_A[i] = Lop
        pair(Lop, Rop, +1.0, "F2", -1.0)
    # F3: for p<q in A:  c†_p c†_q ⊗ P^B_pq  and h.c. (even, +1/+1)
    nA = len(mode_shifts_A)
    o = 0
    for p in range(nA):
        for q in range(p + 1, nA):
            o += 1
            if not keep("F3", o - 1):
                continue
            d = add(mode_shifts_A[p], mode_shifts_A[q])
            Lop = new_op("A", d, 0, False, f"c†c†_{p},{q}")
            Rop = new_op("B", neg(d), 0, False, f"P^B_{p},{q}")
            pair(Lop, Rop, +1.0, "F3", +1.0)
    # F4: for p,s in A:  c†_p c_s ⊗ Q^B_ps ; (s,p) is the h.c. of (p,s)
    o = 0
    for p in range(nA):
        for s in range(p, nA):
            o += 1
            if not keep("F4", o - 1):
                continue
            d = add(mode_shifts_A[p], neg(mode_shifts_A[s]))
            if p == s:
                Lop = new_op("A", zero, 0, True, f"n_{p}")
                Rop = new_op("B", zero, 0, True, f"Q^B_{p},{p}")
                pair(Lop, Rop, +1.0, "F4")
            else:
                Lop = new_op("A", d, 0, False, f"c†c_{p},{s}")
                Rop = new_op("B", neg(d), 0, False, f"Q^B_{p},{s}")
                pair(Lop, Rop, +1.0, "F4", +1.0)
    wl.hermitian = True
    return wl


def spinless_term_structure(n_A, n_B):
    """(mode shifts of A, mode shifts of B) for spinless fermions: one U(1)."""
    return [(1,)] * n_A, [(1,)] * n_B


def hubbard_term_structure(n_orb_A, n_orb_B):
    """Spin-orbital order (site ↑, site ↓, ...) — reading r8; charges (n↑, n↓)."""
    return [(1, 0), (0, 1)] * n_orb_A, [(1, 0), (0, 1)] * n_orb_B


def lattice_workload(kind, n_half, M, seed, name=None, width2=None, keep=None):
    """Configs 3-5 and their scaled-down copies.

    kind = "spinless": n_half modes per half, sectors q=0..n_half,
           w_q = exp(-(q-n_half/2)²/width2), width2 default n_half (σ² = n_half/2:
           32 for the 8×8 half, 72 for the 12×12 half), caps C(n_half, q),
           target N = n_half (half filling of 2·n_half modes).
    kind = "hubbard":  n_half spatial orbitals per half, sectors (n↑,n↓) in
           [0,n_half]², w = exp(-((n↑-c)²+(n↓-c)²)/width2), c = n_half/2,
           width2 default 8·n_half/18 (8 for the 6×6 half), caps
           C(n_half,n↑)·C(n_half,n↓), target (n_half, n_half).
    """
    if kind == "spinless":
        width2 = float(n_half) if width2 is None else width2
        c = n_half / 2.0
        qs = [(q,) for q in range(n_half + 1)]
        w = [math.exp(-((q[0] - c) ** 2) / width2) for q in qs]
        caps = [binom(n_half, q[0]) for q in qs]
        target = (n_half,)
        shifts = spinless_term_structure(n_half, n_half)
    elif kind == "hubbard":
        width2 = 8.0 * n_half / 18.0 if width2 is None else width2
        c = n_half / 2.0
        qs = [(u, d) for u in range(n_half + 1) for d in range(n_half + 1)]
        w = [math.exp(-(((u - c) ** 2) + ((d - c) ** 2)) / width2) for u, d in qs]
        caps = [binom(n_half, u) * binom(n_half, d) for u, d in qs]
        target = (n_half, n_half)
        shifts = hubbard_term_structure(n_half, n_half)
    else:
        raise ValueError(kind)
    dims = gaussian_sectors(M, w, caps)
    sectors = [(q, d) for q, d in zip(qs, dims)]
    wl = Workload(name or f"{kind}_n{n_half}_M{M}", seed, len(target), sectors, list(sectors), target)
    return _family_builder(wl, shifts[0], shifts[1], keep=keep)


# ----------------------------------------------------------------------------
# the BASELINE.json configs by name (configs[0] is real physics and comes from
# the oracle's DMRG, see tests/_gpu.config1_problem)
# ----------------------------------------------------------------------------
def config3():
    """configs[2]: 8×8 spinless torus, mode-rotated, D = 2048 (M = 4096), K = 2146."""
    return lattice_workload("spinless", 32, 4096, seed=3, name="config3_spinless8x8_rotated_D2048")


def config4():
    """configs[3]: 6×6 Hubbard torus, mode-rotated, D = 4096 (M = 16384), K = 2702."""
    return lattice_workload("hubbard", 18, 16384, seed=4, name="config4_hubbard6x6_rotated_D4096")


def config4_realspace():
    """configs[3], real-space variant: on-site U gives no cross-cut two-body
    term, so only H_A, H_B and the hopping of the 12 boundary sites × 2 spins cross the cut:
    K = 2 + 12·2·2 = 50.  Built as the F0 + thinned F1/F2 families of the rotated list."""
    keep = lambda fam, i: fam == "F1" and i < 24
    return lattice_workload("hubbard", 18, 16384, seed=4, name="config4_hubbard6x6_realspace_D4096", keep=keep)


def config5_keep(fam, i):
    """Executed subset of configs[4]: every F1/F2 pair, every 12th F3 and F4 pair (same
    family proportions as a stratified sample of the 10 586-pair list)."""
    return fam in ("F1", "F2") or i % 12 == 0


def config5():
    """configs[4]: 12×12 spinless torus, mode-rotated, D = 8192 (M = 16384).  The full list
    (K = 10 586, ≈ 1.05 TB of operators stored once) cannot fit; the executed subset keeps
    K_exec pairs (≈ 115 GB) of which ``config5_staged_ops`` are bound to pinned host memory."""
    return lattice_workload("spinless", 72, 16384, seed=5, name="config5_spinless12x12_rotated_D8192_subset",
                            keep=config5_keep)


def config5_staged_ops(wl):
    """Every 7th stored operator streams from pinned host memory (≈ 14 % of the bytes)."""
    return [i for i in range(len(wl.ops)) if i % 7 == 3]


# ----------------------------------------------------------------------------
# SU(2) spin-adapted singlet workload: structure only
# ----------------------------------------------------------------------------
def su2_multiplet_count(n_orb, N, two_s):
    """Number of spin-S multiplets with N electrons in n_orb orbitals: dim(S_z = S) − dim(S_z = S + 1)."""
    if (N + two_s) % 2 or two_s < 0:
        return 0
    up, dn = (N + two_s) // 2, (N - two_s) // 2
    c = lambda a, b: binom(n_orb, a) * binom(n_orb, b) if 0 <= a <= n_orb and 0 <= b <= n_orb else 0
    return c(up, dn) - c(up + 1, dn - 1)


def su2_singlet_workload(n_half=18, M=12288, seed=6, name=None, keep=None, width_n=8.0, width_s=6.0):
    """The operator-pair list of a Hubbard-type lattice half with n_half orbitals per side in SPIN-ADAPTED form,
    for a spin-singlet target at half filling — sector structure and term structure only, values synthetic (r17).

    Sectors: A labelled (N, 2S), B labelled (N, −2S) (for total spin 0 both halves of a ψ block carry the same S,
    so the labels add up to the target (2·n_half, 0)); dims count MULTIPLETS, ∝ (2S+1)·exp(−(N−n_half)²/width_n
    − S(S+1)/width_s), capped by the number of multiplets that exist, M in total (M = 3·D: a site has three
    multiplets).  Terms: the families F0-F4 over the orbitals, every rank-k tensor operator stored once per
    Δ(2S) ∈ {−2k … 2k} — which is the U(1)×U(1) list with the two spin components of an orbital replaced by the two
    "virtual modes" of label shift (1, +1) and (1, −1).  ``wl.ranks[k]`` is the doubled tensor rank of pair k (an
    input of the recoupling table): ½ for F1/F2, 1 for the Δ(2S) = ±2 pairs of F3/F4, and of the two Δ(2S) = 0 pairs of
    an orbital pair one is the triplet's and one the singlet's."""
    import re
    qs = []
    for N in range(2 * n_half + 1):
        for two_s in range(N % 2, min(N, 2 * n_half - N) + 1, 2):
            if su2_multiplet_count(n_half, N, two_s) > 0:
                qs.append((N, two_s))
    w = [(t + 1) * math.exp(-((N - n_half) ** 2) / width_n - (t / 2.0) * (t / 2.0 + 1.0) / width_s) for N, t in qs]
    caps = [su2_multiplet_count(n_half, N, t) for N, t in qs]
    dims = gaussian_sectors(M, w, caps)
    sectors_A = [(q, d) for q, d in zip(qs, dims)]
    sectors_B = [((N, -t), d) for (N, t), d in zip(qs, dims)]
    wl = Workload(name or f"su2_singlet_n{n_half}_M{M}", seed, 2, sectors_A, sectors_B, (2 * n_half, 0))
    shifts_A = [(1, 1), (1, -1)] * n_half
    shifts_B = [(1, -1), (1, 1)] * n_half
    _family_builder(wl, shifts_A, shifts_B, keep=keep)
    wl.ranks = []
    for t in wl.terms:
        fam = t.family.replace("^hc", "")
        if fam == "F0":
            wl.ranks.append(0)
        elif fam in ("F1", "F2"):
            wl.ranks.append(1)
        else:
            op = wl.ops[t.L]
            if op.dq[1] != 0:
                wl.ranks.append(abs(op.dq[1]))
            else:
                idx = [int(x) for x in re.findall(r"\d+", op.tag)]
                same_orbital = len(idx) == 2 and idx[0] // 2 == idx[1] // 2 and fam == "F3"
                wl.ranks.append(0 if same_orbital or idx[0] % 2 else 2)
    return wl


def sub_workload(wl, term_ids, name=None):
    """The workload restricted to the operator pairs ``term_ids`` (a shard of the k list):
    same sectors and target, only the stored operators those pairs touch, re-indexed, each keeping the
    RNG stream it has in ``wl`` so that its values are unchanged.  Σ over a partition of the pair list
    of the shards' σ equals the σ of ``wl`` (k-additivity)."""
    import copy
    term_ids = list(term_ids)
    used = sorted({i for k in term_ids for i in (wl.terms[k].L, wl.terms[k].R) if i is not None})
    new_index = {old: new for new, old in enumerate(used)}
    sub = Workload(name or f"{wl.name}_sub{len(term_ids)}", wl.seed, wl.n_charges, list(wl.sectors_A),
                   list(wl.sectors_B), tuple(wl.target), hermitian=False)
    for old in used:
        spec = copy.copy(wl.ops[old])
        spec.stream = op_stream_of(wl, old)
        sub.ops.append(spec)
    for k in term_ids:
        t = copy.copy(wl.terms[k])
        t.L = None if t.L is None else new_index[t.L]
        t.R = None if t.R is None else new_index[t.R]
        sub.terms.append(t)
    return sub


# ----------------------------------------------------------------------------
# renormalisation inputs: the kept basis Φ of half A
# ----------------------------------------------------------------------------
PHI_STREAM = 13


def renorm_basis(wl, M_new=None, half="A"):
    """Sector list of the kept (new) basis of one half of ``wl`` and the block table of Φ.

    The new basis keeps M_new states (default M/d with d = 2 spinless, 4 Hubbard: the bond
    dimension D behind the enlarged dimension M = d·D, reading r9), distributed over the same
    charges by the workload's own sector law (largest-remainder rounding, capped by the enlarged
    dims).  Returns (sectors_new, phi_table) with phi_table = [(enl_idx, new_idx, rows, cols, off)],
    off counting unpadded elements block after block in enlarged-sector order; sectors that keep no
    state are dropped from the new space."""
    sectors = wl.sectors(half)
    M = sum(d for _, d in sectors)
    d_loc = 2 if wl.n_charges == 1 else 4
    M_new = M // d_loc if M_new is None else M_new
    w = [float(d) for _, d in sectors]
    dims = gaussian_sectors(M_new, w, [d for _, d in sectors]) if M_new < M else [d for _, d in sectors]
    sectors_new, table, off = [], [], 0
    for ei, ((q, de), dn) in enumerate(zip(sectors, dims)):
        if dn <= 0 or de <= 0:
            continue
        table.append((ei, len(sectors_new), de, dn, off))
        sectors_new.append((q, dn))
        off += de * dn
    return sectors_new, table


def fill_phi_host(wl, phi_table, stream=PHI_STREAM):
    """Φ blocks {(enl_idx, new_idx): ndarray}: normal12 / sqrt(rows) (synthetic: not orthonormal,
    which the products do not need)."""
    out = {}
    for (ei, ni, rows, cols, off) in phi_table:
        idx = off + np.arange(rows * cols, dtype=np.uint64).reshape(rows, cols)
        out[(ei, ni)] = normal12(wl.seed, stream, idx) * (1.0 / math.sqrt(rows))
    return out
