"""T1: a simple two-site DMRG with explicit Fock-space block bases, and the
definition of the effective Hamiltonian, H_eff = P† H P.

The paper gives no algorithmic detail ("The details of the algorithm can be
found in various review articles"), so this follows the textbook
two-site algorithm in the most literal form possible for ≤ 16-18 modes
(reading T1 of SURVEY.md §8(c), recorded in DESIGN.md):

  * A block basis is an explicit isometry Φ (2^{modes} × D) whose columns have
    definite charges; the MPS of Eq. (4) is implicit in the nesting
    Φ_L[i+1] = (Φ_L[i] ⊗ 1_site) U,  Φ_R[i] = (1_site ⊗ Φ_R[i+1]) V.
  * At bond (i, i+1): A = Φ_L[i] ⊗ 1_site (enlarged left block), B = 1_site ⊗
    Φ_R[i+2] (enlarged right block), both re-ordered sector-major; the two-site
    space is {|a⟩⊗|b⟩ : q_a + q_b = target}; P maps it into Fock space and
    H_eff = P† H P is solved *exactly* with a dense symmetric eigensolver.
  * Truncation: SVD of every charge block of ψ[a,b] separately (an SVD of the
    whole matrix would mix degenerate singular vectors across sectors), then
    keep the D largest singular values globally (ties → lower index).
  * Start: seeded N(0,1)-like vector in the target sector, normalised, turned
    into right bases by successive truncated SVDs from the right; one full
    sweep (→, ←), then → to the requested bond; the hot-call input ψ is the
    current state projected on that bond's two-site space, before optimisation.
"""
from dataclasses import dataclass, field
import numpy as np
import scipy.linalg
import scipy.sparse as sp

from . import fock
from workloads.rng import normal12


@dataclass
class Basis:
    Phi: np.ndarray      # (2^m, D) orthonormal columns
    q: np.ndarray        # (D, n_charges) integer charge of every column
    n_modes: int


def trivial_basis(n_charges):
    return Basis(np.ones((1, 1)), np.zeros((1, n_charges), dtype=np.int64), 0)


def site_basis(mode_charges):
    m = len(mode_charges)
    return Basis(np.eye(2 ** m), fock.charges_of_states(m, mode_charges), m)


def kron_basis(left, right):
    """Product basis, left index major: |l⟩⊗|r⟩ ↦ column l·D_r + r."""
    Phi = np.kron(left.Phi, right.Phi)
    q = (left.q[:, None, :] + right.q[None, :, :]).reshape(-1, left.q.shape[1])
    return Basis(Phi, q, left.n_modes + right.n_modes)


def sector_major(basis):
    """Columns re-ordered sector-major (charges ascending lexicographically,
    stable inside a sector).  Returns (basis, [(charge tuple, dim)])."""
    keys = [tuple(int(x) for x in row) for row in basis.q]
    order = sorted(range(len(keys)), key=lambda i: (keys[i], i))
    b = Basis(basis.Phi[:, order], basis.q[order], basis.n_modes)
    sectors = []
    for i in order:
        if sectors and sectors[-1][0] == keys[i]:
            sectors[-1][1] += 1
        else:
            sectors.append([keys[i], 1])
    return b, [(k, d) for k, d in sectors]


def sector_slices(sectors):
    out, o = [], 0
    for _, d in sectors:
        out.append(slice(o, o + d))
        o += d
    return out


@dataclass
class TwoSiteSpace:
    A: Basis
    B: Basis
    sectors_A: list
    sectors_B: list
    target: tuple
    blocks: list = field(default_factory=list)   # [(ai, bi, rows, cols, offset)] allowed ψ blocks

    @property
    def dim(self):
        return sum(r * c for _, _, r, c, _ in self.blocks)


def two_site_space(A, B, target):
    A, sa = sector_major(A)
    B, sb = sector_major(B)
    idxB = {q: i for i, (q, _) in enumerate(sb)}
    blocks, off = [], 0
    for ai, (qa, da) in enumerate(sa):
        qb = tuple(t - x for t, x in zip(target, qa))
        if qb in idxB:
            bi = idxB[qb]
            blocks.append((ai, bi, da, sb[bi][1], off))
            off += da * sb[bi][1]
    return TwoSiteSpace(A, B, sa, sb, tuple(target), blocks)


def projector(space, fock_rows):
    """P restricted to the Fock rows ``fock_rows``: columns are |a⟩⊗|b⟩ for the
    allowed blocks, block after block, a major inside a block."""
    slA, slB = sector_slices(space.sectors_A), sector_slices(space.sectors_B)
    P = np.zeros((len(fock_rows), space.dim))
    for ai, bi, da, db, off in space.blocks:
        blk = np.kron(space.A.Phi[:, slA[ai]], space.B.Phi[:, slB[bi]])
        P[:, off:off + da * db] = blk[fock_rows]
    return P


def vec_to_blocks(space, x):
    return {(ai, bi): x[off:off + da * db].reshape(da, db) for ai, bi, da, db, off in space.blocks}


def blocks_to_vec(space, blocks):
    x = np.zeros(space.dim)
    for ai, bi, da, db, off in space.blocks:
        x[off:off + da * db] = blocks[(ai, bi)].reshape(-1)
    return x


def truncate(space, x, D):
    """Block-wise SVD of ψ, keep the D largest singular values globally.
    Returns (U, qU, V, qV, discarded weight): columns of U live in A's space
    (M_A × D'), columns of V in B's space (M_B × D')."""
    slA, slB = sector_slices(space.sectors_A), sector_slices(space.sectors_B)
    MA = sum(d for _, d in space.sectors_A)
    MB = sum(d for _, d in space.sectors_B)
    cand = []
    svds = {}
    for ai, bi, da, db, off in space.blocks:
        u, s, vt = np.linalg.svd(x[off:off + da * db].reshape(da, db), full_matrices=False)
        svds[(ai, bi)] = (u, s, vt)
        for j, sv in enumerate(s):
            cand.append((-sv, len(cand), ai, bi, j))
    cand.sort()
    kept = [c for c in cand[:D] if -c[0] > 1e-14]
    kept.sort(key=lambda c: c[1])
    U = np.zeros((MA, len(kept)))
    V = np.zeros((MB, len(kept)))
    qU = np.zeros((len(kept), len(space.target)), dtype=np.int64)
    qV = np.zeros_like(qU)
    for col, (_, _, ai, bi, j) in enumerate(kept):
        u, s, vt = svds[(ai, bi)]
        U[slA[ai], col] = u[:, j]
        V[slB[bi], col] = vt[j, :]
        qU[col] = space.sectors_A[ai][0]
        qV[col] = space.sectors_B[bi][0]
    disc = sum(c[0] ** 2 for c in cand[D:])
    return U, qU, V, qV, disc


def lowest_eigenpair(H):
    w, v = scipy.linalg.eigh(H, subset_by_index=[0, 0])
    return float(w[0]), v[:, 0]


class SimpleDMRG:
    """Two-site DMRG on ≤ ~18 modes with everything explicit in Fock space."""

    def __init__(self, T, V, mode_charges, site_modes, target, D, seed, sector_hamiltonian=False):
        """``sector_hamiltonian``: build H inside the target sector from bit-string actions
        (fock.hamiltonian_sector, pinned against the Kronecker construction) instead of restricting the
        2^n-dimensional Kronecker matrix — same matrix, needed where a dense V makes the latter too slow."""
        self.T, self.V = T, V
        self.mc = np.asarray(mode_charges, dtype=np.int64).reshape(T.shape[0], -1)
        self.n = T.shape[0]
        self.site_modes = site_modes
        self.n_sites = len(site_modes)
        self.target = tuple(int(x) for x in target)
        self.D = D
        self.rows = fock.sector_indices(self.n, self.mc, self.target)
        if sector_hamiltonian:
            rows, self.H = fock.hamiltonian_sector(T, V, self.mc, self.target)
            assert np.array_equal(rows, self.rows)
        else:
            self.H = fock.restrict(fock.hamiltonian(T, V), self.rows).tocsr()
        self.sites = [site_basis(self.mc[m]) for m in site_modes]
        nc = self.mc.shape[1]
        self.L = {0: trivial_basis(nc)}
        self.R = {self.n_sites: trivial_basis(nc)}
        g = normal12(seed, 5, np.arange(len(self.rows)))
        self.state = g / np.linalg.norm(g)          # amplitudes on self.rows
        self.energies = []
        self._init_right_bases()

    # -- start: right bases from successive truncated SVDs of the seed vector
    def _init_right_bases(self):
        full = np.zeros(2 ** self.n)
        full[self.rows] = self.state
        for l in range(self.n_sites - 1, 0, -1):
            Bl, sectors = sector_major(kron_basis(self.sites[l], self.R[l + 1]))
            m_right = Bl.n_modes
            C = full.reshape(2 ** (self.n - m_right), 2 ** m_right) @ Bl.Phi
            cand, svds = [], {}
            for si, sl in enumerate(sector_slices(sectors)):
                u, s, vt = np.linalg.svd(C[:, sl], full_matrices=False)
                svds[si] = (s, vt, sl)
                for j, sv in enumerate(s):
                    cand.append((-sv, len(cand), si, j))
            cand.sort()
            kept = [c for c in cand[:self.D] if -c[0] > 1e-14]
            kept.sort(key=lambda c: c[1])
            Vm = np.zeros((Bl.Phi.shape[1], len(kept)))
            q = np.zeros((len(kept), self.mc.shape[1]), dtype=np.int64)
            for col, (_, _, si, j) in enumerate(kept):
                s, vt, sl = svds[si]
                Vm[sl, col] = vt[j, :]
                q[col] = sectors[si][0]
            self.R[l] = Basis(Bl.Phi @ Vm, q, m_right)

    def space_at(self, i):
        """Two-site space of bond (i, i+1): left block = sites < i, right block = sites > i+1."""
        A = kron_basis(self.L[i], self.sites[i])
        B = kron_basis(self.sites[i + 1], self.R[i + 2])
        return two_site_space(A, B, self.target)

    def heff_at(self, space):
        P = projector(space, self.rows)
        Heff = P.T @ (self.H @ P)
        return 0.5 * (Heff + Heff.T), P

    def guess_at(self, space, P=None):
        """Current state projected on the two-site space (wave-function transformation)."""
        P = projector(space, self.rows) if P is None else P
        x = P.T @ self.state
        return x / np.linalg.norm(x)

    def step(self, i, direction):
        space = self.space_at(i)
        Heff, P = self.heff_at(space)
        E, x = lowest_eigenpair(Heff)
        U, qU, V, qV, _ = truncate(space, x, self.D)
        if direction > 0:
            self.L[i + 1] = Basis(space.A.Phi @ U, qU, space.A.n_modes)
        else:
            self.R[i + 1] = Basis(space.B.Phi @ V, qV, space.B.n_modes)
        # truncated state, renormalised, back in Fock space
        xt = np.zeros_like(x)
        slA, slB = sector_slices(space.sectors_A), sector_slices(space.sectors_B)
        for ai, bi, da, db, off in space.blocks:
            blk = x[off:off + da * db].reshape(da, db)
            xt[off:off + da * db] = (U[slA[ai]] @ (U[slA[ai]].T @ blk @ V[slB[bi]]) @ V[slB[bi]].T).reshape(-1)
        xt /= np.linalg.norm(xt)
        self.state = P @ xt
        self.energies.append(E)
        return E

    def sweep_right(self, start, stop):
        for i in range(start, stop):
            self.step(i, +1)

    def sweep_left(self, start, stop):
        for i in range(start, stop, -1):
            self.step(i, -1)

    def warmup_to(self, bond):
        """One full sweep (→ then ←), then → up to (not including) ``bond``."""
        self.sweep_right(0, self.n_sites - 1)
        self.sweep_left(self.n_sites - 2, -1)     # turning bond re-solved: sets R[n_sites-1]
        self.sweep_right(0, bond)
        return self
