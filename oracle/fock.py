"""T0: Fock-space matrices with Jordan-Wigner signs and exact diagonalisation.

Conventions (used by every oracle tier):
  * n modes ordered along the MPS chain, mode 0 first.
  * Basis state |n_0 n_1 … n_{n-1}⟩ = (c†_0)^{n_0} (c†_1)^{n_1} … |vac⟩ has index
    Σ_p n_p 2^{n-1-p} (mode 0 is the most significant bit), i.e. the Kronecker
    order of np.kron(factor_0, factor_1, …).
  * c_p = Z ⊗ … ⊗ Z ⊗ a ⊗ 1 ⊗ … ⊗ 1 with p factors Z = diag(1,−1) and
    a = |0⟩⟨1|, so c_p |…n_p…⟩ = (−1)^{Σ_{q<p} n_q} n_p |…0_p…⟩, which gives the
    canonical anticommutation relations quoted at PAPER.md:68.
  * Eq. (1) is taken literally, with no ½ prefactor:
    H = Σ_ij T_ij c†_i c_j + Σ_ijkl V_ijkl c†_i c†_j c_k c_l ; the (generalised)
    spin index of the paper is folded into the mode index.
"""
import numpy as np
import scipy.sparse as sp

_A = sp.csr_matrix(np.array([[0.0, 1.0], [0.0, 0.0]]))
_Z = sp.csr_matrix(np.array([[1.0, 0.0], [0.0, -1.0]]))


def annihilators(n):
    """[c_0 … c_{n-1}] as sparse 2^n × 2^n matrices (Jordan-Wigner)."""
    ops = []
    for p in range(n):
        m = sp.identity(1, format="csr")
        for q in range(n):
            f = _Z if q < p else (_A if q == p else sp.identity(2, format="csr"))
            m = sp.kron(m, f, format="csr")
        ops.append(m)
    return ops


def occupations(n):
    """(2^n × n) integer array: occupations[index, p] = n_p of basis state index."""
    idx = np.arange(2 ** n, dtype=np.int64)
    return np.stack([(idx >> (n - 1 - p)) & 1 for p in range(n)], axis=1) if n else np.zeros((1, 0), np.int64)


def charges_of_states(n, mode_charges):
    """Charge vector of every basis state: occupations @ mode_charges.

    ``mode_charges`` is (n × n_charges): (1,) per mode for spinless fermions,
    (1,0)/(0,1) for ↑/↓ spin-orbitals of the Hubbard model.
    """
    mc = np.asarray(mode_charges, dtype=np.int64).reshape(n, -1)
    return occupations(n) @ mc


def sector_indices(n, mode_charges, target):
    """Indices of the basis states whose charge vector equals ``target``."""
    q = charges_of_states(n, mode_charges)
    return np.nonzero(np.all(q == np.asarray(target, dtype=np.int64), axis=1))[0]


def one_body(T, c=None):
    """Σ_ij T_ij c†_i c_j (sparse)."""
    n = T.shape[0]
    c = annihilators(n) if c is None else c
    H = sp.csr_matrix((2 ** n, 2 ** n))
    for i in range(n):
        ci_dag = c[i].T.tocsr()
        for j in range(n):
            if T[i, j] != 0.0:
                H = H + T[i, j] * (ci_dag @ c[j])
    return H


def two_body(V, c=None):
    """Σ_ijkl V_ijkl c†_i c†_j c_k c_l (sparse), Eq. (1) second sum."""
    n = V.shape[0]
    c = annihilators(n) if c is None else c
    H = sp.csr_matrix((2 ** n, 2 ** n))
    nz = np.argwhere(V != 0.0)
    cache_cc, cache_aa = {}, {}
    for i, j, k, l in nz:
        if i == j or k == l:
            continue  # c†_i c†_i = 0, c_k c_k = 0
        if (i, j) not in cache_cc:
            cache_cc[(i, j)] = (c[i].T @ c[j].T).tocsr()
        if (k, l) not in cache_aa:
            cache_aa[(k, l)] = (c[k] @ c[l]).tocsr()
        H = H + V[i, j, k, l] * (cache_cc[(i, j)] @ cache_aa[(k, l)])
    return H


def hamiltonian(T, V, c=None):
    """Eq. (1) as a sparse 2^n × 2^n matrix."""
    n = T.shape[0]
    c = annihilators(n) if c is None else c
    return (one_body(T, c) + two_body(V, c)).tocsr()


def restrict(H, idx):
    """H restricted to the basis states ``idx`` (rows and columns)."""
    H = H.tocsr()
    return H[idx][:, idx]


def ground_energy(T, V, mode_charges, target, dense_limit=6000):
    """Lowest eigenvalue of Eq. (1) in the charge sector ``target``."""
    n = T.shape[0]
    H = restrict(hamiltonian(T, V), sector_indices(n, mode_charges, target))
    if H.shape[0] <= dense_limit:
        return float(np.linalg.eigvalsh(H.toarray())[0])
    from scipy.sparse.linalg import eigsh
    return float(np.sort(eigsh(H, k=4, which="SA", tol=1e-12, ncv=64)[0])[0])


# ----------------------------------------------------------------------------
# independent brute force: action of an operator string on bit strings
# (shares nothing with the Kronecker construction above; used only as a pin)
# ----------------------------------------------------------------------------
def apply_string_bits(string, occ):
    """Apply a string of ladder operators to one occupation tuple.

    ``string`` is a sequence of (kind, mode), kind '+' for c† and '-' for c,
    written left to right as in the formula, so the *rightmost* acts first.
    Returns (sign, new_occupations) or (0, None).
    """
    occ = list(occ)
    sign = 1
    for kind, p in reversed(list(string)):
        if kind == "-":
            if occ[p] == 0:
                return 0, None
            occ[p] = 0
        else:
            if occ[p] == 1:
                return 0, None
            occ[p] = 1
        if sum(occ[:p]) % 2:
            sign = -sign
    return sign, tuple(occ)


def hamiltonian_bits(T, V):
    """Eq. (1) as a dense matrix, built state by state from ``apply_string_bits``."""
    n = T.shape[0]
    dim = 2 ** n
    occ = occupations(n)
    index = {tuple(o): i for i, o in enumerate(occ.tolist())}
    H = np.zeros((dim, dim))
    for col in range(dim):
        o = tuple(occ[col].tolist())
        for i in range(n):
            for j in range(n):
                if T[i, j] != 0.0:
                    s, new = apply_string_bits([("+", i), ("-", j)], o)
                    if s:
                        H[index[new], col] += s * T[i, j]
        for i, j, k, l in np.argwhere(V != 0.0):
            s, new = apply_string_bits([("+", i), ("+", j), ("-", k), ("-", l)], o)
            if s:
                H[index[new], col] += s * V[i, j, k, l]
    return H


# ----------------------------------------------------------------------------
# Eq. (1) inside one charge sector, for lattices whose 2^n × 2^n matrix with a dense V is out of reach
# (the mode-rotated 4×4 torus: 16⁴ products of 65536-dimensional sparse matrices).  Built from the
# bit-string action of operator strings on the sector's basis states — the construction of the pin above,
# vectorised over states — so it shares nothing with the Kronecker matrices of `annihilators`.
# ----------------------------------------------------------------------------
def sector_action(string, n, cols):
    """The operator string (as in `apply_string_bits`) applied to the basis states ``cols`` (Fock indices):
    sparse 2^n × len(cols) matrix with entry sign at (index of the new state, position of the old one)."""
    occ = np.stack([(cols >> (n - 1 - p)) & 1 for p in range(n)], axis=1).astype(np.int64)
    sign = np.ones(len(cols), dtype=np.int64)
    for kind, p in reversed(list(string)):
        want = 1 if kind == "-" else 0
        sign = np.where(occ[:, p] == want, sign, 0)
        occ[:, p] = 1 - want
        odd = occ[:, :p].sum(axis=1) & 1
        sign = np.where(odd == 1, -sign, sign)
    new = occ @ (1 << np.arange(n - 1, -1, -1, dtype=np.int64))
    keep = sign != 0
    return sp.csr_matrix((sign[keep].astype(np.float64), (new[keep], np.nonzero(keep)[0])), shape=(2 ** n, len(cols)))


def hamiltonian_sector(T, V, mode_charges, target):
    """(rows, H): Eq. (1) (no ½) restricted to the basis states ``rows`` of charge ``target``.

    Σ_ij T_ij c†_i c_j = Σ_ij T_ij (c_i)ᵀ c_j and Σ_ijkl V_ijkl c†_i c†_j c_k c_l = Σ_kl [Σ_ij V_ijkl (c_j c_i)]ᵀ (c_k c_l),
    with c_j and c_k c_l taken as maps from the sector into the full Fock index range; terms that would leave
    the sector are absent because Hᵀ-side and H-side intermediate states must coincide."""
    n = T.shape[0]
    rows = sector_indices(n, mode_charges, target)
    a = [sector_action([("-", j)], n, rows) for j in range(n)]
    H = sp.csr_matrix((len(rows), len(rows)))
    for i in range(n):
        M = None
        for j in range(n):
            if T[i, j] != 0.0:
                M = T[i, j] * a[j] if M is None else M + T[i, j] * a[j]
        if M is not None:
            H = H + a[i].T @ M
    pairs = [(k, l) for k in range(n) for l in range(n) if k != l]
    A = {kl: sector_action([("-", kl[0]), ("-", kl[1])], n, rows).tocoo() for kl in pairs}
    for (k, l) in pairs:
        data, r, c = [], [], []
        for (i, j) in pairs:
            v = V[i, j, k, l]
            if v != 0.0:
                m = A[(j, i)]                    # c†_i c†_j = (c_j c_i)†
                data.append(v * m.data)
                r.append(m.row)
                c.append(m.col)
        if data:
            M = sp.csr_matrix((np.concatenate(data), (np.concatenate(r), np.concatenate(c))), shape=(2 ** n, len(rows)))
            H = H + M.T @ A[(k, l)].tocsr()
    return rows, H.tocsr()
