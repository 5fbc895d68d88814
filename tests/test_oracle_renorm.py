"""Pins of oracle/renorm.py (O′ = Φ† O Φ, "Ren_l / Ren_r")."""
import numpy as np

import workloads as wlmod
from oracle import renorm, heff, lattice, dmrg, export, terms as terms_mod


def _small():
    wl = wlmod.lattice_workload("spinless", 5, 24, seed=3)
    sectors_new, table = wlmod.renorm_basis(wl, M_new=11)
    phi = wlmod.fill_phi_host(wl, table)
    ops = [{"half": s.half, "dq": tuple(s.dq), "parity": s.parity, "blocks": wlmod.fill_op_host(wl, i)}
           for i, s in enumerate(wl.ops) if s.half == "A"]
    return wl, sectors_new, table, phi, ops


def test_recipe_of_the_new_basis():
    wl, sectors_new, table, phi, _ = _small()
    assert sum(d for _, d in sectors_new) == 11
    enl = dict((q, d) for q, d in wl.sectors_A)
    assert all(1 <= d <= enl[q] for q, d in sectors_new)
    assert [t[1] for t in table] == list(range(len(sectors_new)))
    assert all(phi[(e, n)].shape == (r, c) for (e, n, r, c, _) in table)
    big = wlmod.config4()
    sn, tb = wlmod.renorm_basis(big)
    assert sum(d for _, d in sn) == 4096          # D = M/4 for the Hubbard half (reading r9)


def test_blockwise_equals_dense_definition_and_brute_force():
    wl, sectors_new, table, phi, ops = _small()
    off_n, Mn = heff.sector_offsets(sectors_new)
    P = renorm.densify_phi(phi, wl.sectors_A, sectors_new)
    for op in ops[:8]:
        D = renorm.renormalise_dense(op, wl.sectors_A, phi, sectors_new)
        B = renorm.renormalise_blockwise(op, wl.sectors_A, phi, sectors_new)
        R = np.zeros_like(D)
        for (rn, cn), blk in B.items():
            R[off_n[rn]:off_n[rn] + blk.shape[0], off_n[cn]:off_n[cn] + blk.shape[1]] = blk
        assert np.abs(R - D).max() <= 1e-13 * max(1.0, np.abs(D).max())
    # brute force on the element formula O′[i,j] = Σ_ab Φ[a,i] O[a,b] Φ[b,j]
    O = heff.densify_op(ops[2], wl.sectors_A)
    D = renorm.renormalise_dense(ops[2], wl.sectors_A, phi, sectors_new)
    for (i, j) in [(0, 0), (3, 7), (10, 2), (5, 5)]:
        s = 0.0
        for a in range(O.shape[0]):
            for b in range(O.shape[1]):
                s += P[a, i] * O[a, b] * P[b, j]
        assert abs(s - D[i, j]) <= 1e-13 * max(1.0, abs(s))


def test_identity_orthogonal_and_product_rule():
    wl, _, _, _, ops = _small()
    sec = wl.sectors_A
    ident = {(i, i): np.eye(d) for i, (_, d) in enumerate(sec)}
    for op in ops[:5]:
        B = renorm.renormalise_blockwise(op, sec, ident, sec)
        assert set(B) == set(op["blocks"]) and all(np.array_equal(B[k], op["blocks"][k]) for k in B)
    rng = np.random.default_rng(7)
    orth = {(i, i): np.linalg.qr(rng.standard_normal((d, d)))[0] for i, (_, d) in enumerate(sec)}
    sym = next(o for o in ops if all(x == 0 for x in o["dq"]))                # H_A: symmetric blocks
    e0 = np.linalg.eigvalsh(heff.densify_op(sym, sec))
    e1 = np.linalg.eigvalsh(renorm.renormalise_dense(sym, sec, orth, sec))
    assert np.abs(e0 - e1).max() <= 1e-12 * max(1.0, np.abs(e0).max())      # similarity transform
    A, B = heff.densify_op(ops[2], sec), heff.densify_op(ops[3], sec)
    Q = renorm.densify_phi(orth, sec, sec)
    lhs = renorm.renormalise_dense(ops[2], sec, orth, sec) @ renorm.renormalise_dense(ops[3], sec, orth, sec)
    assert np.abs(lhs - Q.T @ (A @ B) @ Q).max() <= 1e-12 * max(1.0, np.abs(A @ B).max())
    # transposition commutes with the map
    t = {"half": "A", "dq": tuple(-x for x in ops[2]["dq"]), "parity": ops[2]["parity"],
         "blocks": {(c, r): b.T.copy() for (r, c), b in ops[2]["blocks"].items()}}
    assert np.abs(renorm.renormalise_dense(t, sec, orth, sec) - renorm.renormalise_dense(ops[2], sec, orth, sec).T).max() < 1e-13


def test_dmrg_bond_operators_carried_by_the_svd_basis():
    """Physics pin: at a bond of the 3×3 spinless torus the exported enlarged-block operators
    L_k = Φ_A† X_k Φ_A, renormalised with the SVD basis U of that bond (Φ_new = Φ_A U), equal
    Φ_new† X_k Φ_new built directly from the Fock-space matrices X_k."""
    T, V, mc = lattice.spinless_tV(3)
    d = dmrg.SimpleDMRG(T, V, mc, [[i] for i in range(9)], (4,), D=6, seed=5)
    d.warmup_to(3)
    space = d.space_at(3)
    pb = export.export_bond(d, space, use_transpose_pairs=False, identity_as_none=False)
    tms = terms_mod.complementary_terms(d.T, d.V, space.A.n_modes, d.mc)
    PhiA = space.A.Phi
    d.step(3, +1)
    new, sectors_new = dmrg.sector_major(d.L[4])
    assert sum(dn for _, dn in sectors_new) <= 6 < PhiA.shape[1]              # a real truncation
    U = PhiA.T @ new.Phi                                                      # M_enl × M_new, sector-major both sides
    assert np.abs(PhiA @ U - new.Phi).max() < 1e-12
    idx_enl = {q: i for i, (q, _) in enumerate(space.sectors_A)}
    sl_e, sl_n = dmrg.sector_slices(space.sectors_A), dmrg.sector_slices(sectors_new)
    phi = {(idx_enl[q], ni): U[sl_e[idx_enl[q]], sl_n[ni]] for ni, (q, _) in enumerate(sectors_new)}
    assert np.abs(renorm.densify_phi(phi, space.sectors_A, sectors_new) - U).max() < 1e-12   # Φ is charge-block diagonal
    a_ops = [o for o in pb.ops if o["half"] == "A"]
    assert len(a_ops) == len(tms)
    worst = 0.0
    for op, t in zip(a_ops, tms):
        direct = new.Phi.T @ (t.X @ new.Phi)
        worst = max(worst, np.abs(renorm.renormalise_dense(op, space.sectors_A, phi, sectors_new) - direct).max())
        B = renorm.renormalise_blockwise(op, space.sectors_A, phi, sectors_new)
        off_n, _ = heff.sector_offsets(sectors_new)
        for (rn, cn), blk in B.items():
            ref = direct[off_n[rn]:off_n[rn] + blk.shape[0], off_n[cn]:off_n[cn] + blk.shape[1]]
            worst = max(worst, np.abs(blk - ref).max())
    assert worst <= 1e-12
