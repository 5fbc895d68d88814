"""T0 inputs: the paper's lattice Hamiltonians as (T, V) of Eq. (1), and mode rotation.

Readings (DESIGN.md table):
  r1  hopping signs follow BASELINE.json: H = −tΣ_nn(c†c+h.c.) − t′Σ_nnn(c†c+h.c.)
      + VΣ_nn n_i n_j   (Eq. (3) prints +t; the sign of t is a gauge on
      the bipartite torus, the sign of t′ is not).
  r2  Eq. (2) is garbled; the Hubbard model is
      −tΣ_⟨ij⟩σ(c†_iσ c_jσ + h.c.) + UΣ_i n_i↑ n_i↓.
  r3  torus bond lists: per site (r,c): nn → (r,c+1), (r+1,c); nnn → (r+1,c+1),
      (r+1,c−1); indices mod L; no de-duplication; each listed bond contributes
      (c†_i c_j + h.c.) once and V n_i n_j once.
  r4  "row-major snake ordering": chain position of (r,c) = r·L + (c if r even
      else L−1−c), 0-based.
  r5  no ½ in Eq. (1): V_ijji = V per listed bond gives V n_i n_j;
      V_{(i↑)(i↓)(i↓)(i↑)} = U gives U n_i↑ n_i↓.
  r6  mode rotation (c_i = Σ_j U_ij d_j, real orthogonal U):
      T′ = Uᵀ T U,  V′_abcd = Σ U_ia U_jb U_kc U_ld V_ijkl.
  r8  Hubbard spin-orbital order: (site 0 ↑, site 0 ↓, site 1 ↑, …).
"""
import numpy as np
import scipy.linalg

from workloads.rng import normal12


def snake_position(r, c, L):
    return r * L + (c if r % 2 == 0 else L - 1 - c)


def torus_bonds(L, order="snake"):
    """(nn, nnn) bond lists between chain positions on an L×L torus (r3, r4)."""
    pos = (lambda r, c: snake_position(r % L, c % L, L)) if order == "snake" \
        else (lambda r, c: (r % L) * L + (c % L))
    nn, nnn = [], []
    for r in range(L):
        for c in range(L):
            i = pos(r, c)
            nn.append((i, pos(r, c + 1)))
            nn.append((i, pos(r + 1, c)))
            nnn.append((i, pos(r + 1, c + 1)))
            nnn.append((i, pos(r + 1, c - 1)))
    return nn, nnn


def spinless_tV(L, t=1.0, tp=0.4, V=0.8, order="snake"):
    """(T, Vtensor, mode_charges) of the t-t′-V model, Eq. (3) with reading r1."""
    n = L * L
    nn, nnn = torus_bonds(L, order)
    T = np.zeros((n, n))
    W = np.zeros((n, n, n, n))
    for i, j in nn:
        T[i, j] += -t
        T[j, i] += -t
        W[i, j, j, i] += V          # c†_i c†_j c_j c_i = n_i n_j  (i ≠ j)
    for i, j in nnn:
        T[i, j] += -tp
        T[j, i] += -tp
    return T, W, np.ones((n, 1), dtype=np.int64)


def hubbard_tV(L, t=1.0, U=4.0, order="snake", bonds=None, n_sites=None):
    """(T, Vtensor, mode_charges) of the Hubbard model (r2, r8).

    ``bonds`` overrides the torus bond list (used for the two-site dimer pin).
    """
    if bonds is None:
        bonds, _ = torus_bonds(L, order)
        n_sites = L * L
    n = 2 * n_sites
    T = np.zeros((n, n))
    W = np.zeros((n, n, n, n))
    for i, j in bonds:
        for s in (0, 1):
            T[2 * i + s, 2 * j + s] += -t
            T[2 * j + s, 2 * i + s] += -t
    for i in range(n_sites):
        up, dn = 2 * i, 2 * i + 1
        W[up, dn, dn, up] += U      # c†_↑ c†_↓ c_↓ c_↑ = n_↑ n_↓
    mc = np.zeros((n, 2), dtype=np.int64)
    mc[0::2, 0] = 1
    mc[1::2, 1] = 1
    return T, W, mc


def rotation_matrix(n, seed, std=0.1, stream=3):
    """U = exp(A), A antisymmetric with A_ij (i<j, row-major) = std·g, g from the
    seeded stream (r6; "entries N(0,0.1)" of BASELINE.json read as std 0.1)."""
    A = np.zeros((n, n))
    iu = np.triu_indices(n, 1)
    g = normal12(seed, stream, np.arange(len(iu[0])))
    A[iu] = std * g
    A = A - A.T
    U = scipy.linalg.expm(A)
    assert np.abs(U.T @ U - np.eye(n)).max() < 1e-13
    return U


def rotate(T, V, U):
    """T′ = Uᵀ T U, V′_abcd = Σ_ijkl U_ia U_jb U_kc U_ld V_ijkl (r6)."""
    Tr = U.T @ T @ U
    Vr = np.einsum("ia,jb,kc,ld,ijkl->abcd", U, U, U, U, V, optimize=True)
    return Tr, Vr


def spin_rotation(U):
    """Same spatial U for both spins, in the (↑,↓)-interleaved order."""
    n = U.shape[0]
    U2 = np.zeros((2 * n, 2 * n))
    U2[0::2, 0::2] = U
    U2[1::2, 1::2] = U
    return U2
