"""-m gpu: one DMRG bond step on the device ("Ren_l"):
the operators of the enlarged left block at bond i are renormalised with the kept basis of that bond
(dmrgk_renorm, O′ = Φᵀ O Φ), the next bond's enlarged-block operators are formed from them and the
site operators (dmrgk_enlarge with the product lists of blockops — including the S^{A′}_p accumulation
and the H_{A′} coupling), and the next bond's σ = H_eff ψ is applied with those operators.
Checked against the oracle's DEFINITIONS: every formed operator against Φ_{A′}† O Φ_{A′} built from
Fock-space matrices (1e-11), and σ against P†HP ψ of the next bond (1e-11).  Truncation (the SVD) is the
oracle's: it is outside the path."""
import numpy as np
import pytest

from oracle import dmrg, terms as oterms, heff
from test_oracle_enlarge import spinless_3x3, hubbard_ring, fock_operator_set
from _gpu import rel_max, TOL_SIGMA

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def cut_blocks(M, sectors_r, sectors_c, dq, same_space=True):
    """Blocks {(row sector idx, col sector idx): array} of a dense matrix for an operator of shift dq."""
    index = {q: i for i, (q, _) in enumerate(sectors_r)}
    sl_r, sl_c = dmrg.sector_slices(sectors_r), dmrg.sector_slices(sectors_c)
    out, mask = {}, np.zeros(M.shape, dtype=bool)
    for ci, (q, dc) in enumerate(sectors_c):
        r = index.get(tuple(a + b for a, b in zip(q, dq)))
        if r is None or dc == 0 or sectors_r[r][1] == 0:
            continue
        out[(r, ci)] = M[sl_r[r], sl_c[ci]].copy()
        mask[sl_r[r], sl_c[ci]] = True
    assert np.abs(M[~mask]).max(initial=0.0) < 1e-11
    return out


class DeviceOps:
    """A set of operators on one space, in one device arena (marshalling only)."""

    def __init__(self, ctx, space, specs, device):
        from paper_2311_14106_b200 import dmrgk
        self.ops = [dmrgk.Op(ctx, space, dq, par) for dq, par in specs]
        total = sum(o.n_padded for o in self.ops)
        self.arena = torch.zeros(max(total, 16), dtype=torch.float64, device=device)
        self.views, o = [], 0
        for op in self.ops:
            v = self.arena[o:o + op.n_padded] if op.n_padded else self.arena[0:16]
            op.bind_device(v)
            self.views.append(v)
            o += op.n_padded

    def upload(self, i, blocks):
        from paper_2311_14106_b200.problem import _unpadded_from_blocks
        op = self.ops[i]
        if op.n_padded:
            self.views[i][:op.n_padded].copy_(torch.from_numpy(op.pack(_unpadded_from_blocks(op.blocks(), blocks))))

    def download(self, i):
        from paper_2311_14106_b200 import dmrgk
        op = self.ops[i]
        r, c, rows, cols, ld, off = op.blocks()
        host = self.views[i].cpu().numpy()
        out, pad_ok = {}, True
        for b in range(len(r)):
            blk = host[off[b]:off[b] + dmrgk.block_size(rows[b], cols[b])]
            out[(int(r[b]), int(c[b]))] = dmrgk.block_unpack(blk, rows[b], cols[b])
            pad_ok = pad_ok and dmrgk.block_padding_is_zero(blk, rows[b], cols[b])
        return out, pad_ok


@pytest.mark.parametrize("make,bond", [(spinless_3x3(64), 3), (spinless_3x3(6), 3), (hubbard_ring(16), 0)])
def test_bond_step_on_the_device(make, bond):
    from paper_2311_14106_b200 import dmrgk, blockops, problem
    T, V, mc, site_modes, target, D = make
    d = dmrg.SimpleDMRG(T, V, mc, site_modes, target, D=D, seed=2)
    d.warmup_to(bond)
    space = d.space_at(bond)                                   # bond i: A = enlarged left block
    A = [m for s in site_modes[:bond + 1] for m in s]
    S = list(site_modes[bond + 1])
    right = [m for s in site_modes[bond + 2:] for m in s]
    keys_A = blockops.left_block_keys(A, S + right)
    XA = fock_operator_set(T, V, mc, len(A))
    d.step(bond, +1)                                           # the oracle's truncation → kept basis of A
    kept, sectors_K = dmrg.sector_major(d.L[bond + 1])
    assert np.array_equal(kept.Phi, d.L[bond + 1].Phi)         # already sector-major (in A's sector order)
    U = space.A.Phi.T @ kept.Phi                               # kept basis in the enlarged basis of A

    dev = torch.device("cuda", 0)
    ctx = dmrgk.Ctx(0)
    nc = d.mc.shape[1]
    sp_A = dmrgk.Space(ctx, nc, space.sectors_A)
    sp_K = dmrgk.Space(ctx, nc, sectors_K)
    # ---- operators of A at bond i (the L_k of that bond), uploaded ----
    specs_A = [blockops.operator_spec(k, mc) for k in keys_A]
    ops_A = DeviceOps(ctx, sp_A, specs_A, dev)
    for i, k in enumerate(keys_A):
        ops_A.upload(i, cut_blocks(space.A.Phi.T @ (XA[k] @ space.A.Phi), space.sectors_A, space.sectors_A, specs_A[i][0]))
    # ---- renormalise: O′ = Φᵀ O Φ ----
    phi = dmrgk.Iso(ctx, sp_A, sp_K)
    pr, pc, prow, pcol, _, _ = phi.blocks()
    slA, slK = dmrg.sector_slices(space.sectors_A), dmrg.sector_slices(sectors_K)
    phi_blocks = {(int(pr[b]), int(pc[b])): U[slA[pr[b]], slK[pc[b]]] for b in range(len(pr))}
    phi_arena = torch.zeros(max(phi.n_padded, 16), dtype=torch.float64, device=dev)
    phi_arena[:phi.n_padded].copy_(torch.from_numpy(phi.pack(problem._unpadded_from_blocks(phi.blocks(), phi_blocks))))
    phi.bind_device(phi_arena)
    ops_K = DeviceOps(ctx, sp_K, specs_A, dev)
    plan = dmrgk.Renorm(ctx, phi, ops_A.ops, ops_K.ops)
    ws = torch.empty(max(plan.workspace_bytes, 128), dtype=torch.uint8, device=dev)
    plan.apply(ws, torch.cuda.current_stream())
    # ---- enlarge: operators of A′ = kept ⊗ site ----
    site, lists = blockops.enlarge_left_lists(T, V, mc, A, S, right)
    space2 = d.space_at(bond + 1)                              # bond i+1: A′ | B′
    keys_Ap = blockops.left_block_keys(A + S, right)
    specs_Ap = [blockops.operator_spec(k, mc) for k in keys_Ap]
    sp_E = dmrgk.Space(ctx, nc, space2.sectors_A)
    ops_E = DeviceOps(ctx, sp_E, specs_Ap, dev)
    ops_E.arena.fill_(float("nan"))                            # enlarge_apply must overwrite everything
    index_K = {k: i for i, k in enumerate(keys_A)}
    terms = []
    for o, key in enumerate(keys_Ap):
        for (k, tr, y, pi) in lists[key]:
            terms.append((o, None if k is None else ops_K.ops[index_K[k]], tr, bool(pi), 1.0, y))
    enl = dmrgk.Enlarge(ctx, sp_K, sp_E, site.charges, ops_E.ops, terms)
    enl.apply(torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert enl.n_tiles > 0 and enl.bytes_read > 0
    # ---- every formed operator against its definition Φ_{A′}† O Φ_{A′} ----
    XAp = fock_operator_set(T, V, mc, len(A) + len(S))
    for i, key in enumerate(keys_Ap):
        ref = cut_blocks(space2.A.Phi.T @ (XAp[key] @ space2.A.Phi), space2.sectors_A, space2.sectors_A, specs_Ap[i][0])
        got, pad_ok = ops_E.download(i)
        assert pad_ok and set(got) == set(ref), key
        scale = max(1.0, max((np.abs(v).max() for v in ref.values() if v.size), default=1.0))
        err = max((np.abs(got[k] - ref[k]).max() for k in ref if ref[k].size), default=0.0)
        assert err <= 1e-11 * scale, (key, err)
    # ---- the next bond's σ with the device-formed L operators ----
    Heff, P = d.heff_at(space2)
    x = d.guess_at(space2, P)
    n_Ap = len(A) + len(S)
    ops, tms = [], []
    index_E = {k: i for i, k in enumerate(keys_Ap)}
    for key in keys_Ap:
        dq, par = blockops.operator_spec(key, mc)
        ops.append({"half": "A", "dq": dq, "parity": par, "blocks": {}})
    for t in oterms.complementary_terms(T, V, n_Ap, mc, prune=False):
        fam, lab = t.family, tuple(t.label)
        Lk, tL = {"F1": (("S",) + lab, False), "F1h": (("S",) + lab, True), "F2": (("c+",) + lab, False),
                  "F2h": (("c+",) + lab, True), "F3": (("c+c+",) + lab, False), "F3h": (("c+c+",) + lab, True)}.get(fam, (None, False))
        if fam == "F0":
            Lk = ("H",) if lab == ("A",) else None
        if fam == "F4":
            Lk, tL = (("c+c",) + lab, False) if lab[0] <= lab[1] else (("c+c", lab[1], lab[0]), True)
        Ri = None
        if not (fam == "F0" and lab == ("A",)):
            Yd = space2.B.Phi.T @ (t.Y @ space2.B.Phi)
            neg = tuple(-v for v in t.dq_A)
            ops.append({"half": "B", "dq": neg, "parity": t.parity, "blocks": cut_blocks(Yd, space2.sectors_B, space2.sectors_B, neg)})
            Ri = len(ops) - 1
        tms.append((None if Lk is None else index_E[Lk], Ri, t.coef, tL, False))
    dp = problem.DeviceProblem(nc, space2.sectors_A, space2.sectors_B, space2.target, ctx=ctx)
    dp.create_ops([(o["half"], o["dq"], o["parity"]) for o in ops])
    dp.alloc_resident()
    for i, o in enumerate(ops):
        if o["half"] == "B":
            dp.set_op_host(i, o["blocks"])
        elif dp.ops[i].n_padded:
            assert dp.ops[i].n_padded == ops_E.ops[i].n_padded
            dp.op_views[i].copy_(ops_E.views[i][:dp.ops[i].n_padded])       # the device-formed operator, as is
    dp.build(tms)
    sigma = dp.to_blocks(dp.apply(dp.psi_from_host(dmrg.vec_to_blocks(space2, x))))
    assert rel_max(sigma, dmrg.vec_to_blocks(space2, Heff @ x)) <= TOL_SIGMA


@pytest.mark.parametrize("make,bond", [(spinless_3x3(64), 4), (spinless_3x3(6), 4), (hubbard_ring(16), 2)])
def test_left_moving_bond_step_right_block_with_S_P_Q(make, bond):
    """The mirror step of a right-to-left sweep: the right block's operators (H_B, c†_p and the
    complementary S^B_p, P^B_pq, Q^B_ps) are renormalised with the kept basis of B, then B′ = site ⊗ B is
    formed on the device — the S, P, Q accumulations of blockops.enlarge_right_lists — and the previous
    bond's σ is applied with them as R operators."""
    from paper_2311_14106_b200 import dmrgk, blockops, problem
    from test_oracle_enlarge import fock_right_set
    T, V, mc, site_modes, target, D = make
    d = dmrg.SimpleDMRG(T, V, mc, site_modes, target, D=D, seed=2)
    d.warmup_to(bond)
    space = d.space_at(bond)                                   # bond i: B = enlarged right block
    left = [m for s in site_modes[:bond] for m in s]
    S = list(site_modes[bond])
    B = [m for s in site_modes[bond + 1:] for m in s]
    n_A = len(left) + len(S)
    keys_B = blockops.right_block_keys(B, left + S)
    YB = fock_right_set(T, V, mc, n_A)
    d.step(bond, -1)
    kept, sectors_K = dmrg.sector_major(d.R[bond + 1])
    U = space.B.Phi.T @ kept.Phi
    dev = torch.device("cuda", 0)
    ctx = dmrgk.Ctx(0)
    nc = d.mc.shape[1]
    sp_B = dmrgk.Space(ctx, nc, space.sectors_B)
    sp_K = dmrgk.Space(ctx, nc, sectors_K)
    specs_B = [blockops.right_operator_spec(k, mc) for k in keys_B]
    ops_B = DeviceOps(ctx, sp_B, specs_B, dev)
    for i, k in enumerate(keys_B):
        ops_B.upload(i, cut_blocks(space.B.Phi.T @ (YB[k] @ space.B.Phi), space.sectors_B, space.sectors_B, specs_B[i][0]))
    phi = dmrgk.Iso(ctx, sp_B, sp_K)
    pr, pc, _, _, _, _ = phi.blocks()
    slB, slK = dmrg.sector_slices(space.sectors_B), dmrg.sector_slices(sectors_K)
    phi_blocks = {(int(pr[b]), int(pc[b])): U[slB[pr[b]], slK[pc[b]]] for b in range(len(pr))}
    phi_arena = torch.zeros(max(phi.n_padded, 16), dtype=torch.float64, device=dev)
    phi_arena[:phi.n_padded].copy_(torch.from_numpy(phi.pack(problem._unpadded_from_blocks(phi.blocks(), phi_blocks))))
    phi.bind_device(phi_arena)
    ops_K = DeviceOps(ctx, sp_K, specs_B, dev)
    plan = dmrgk.Renorm(ctx, phi, ops_B.ops, ops_K.ops)
    ws = torch.empty(max(plan.workspace_bytes, 128), dtype=torch.uint8, device=dev)
    plan.apply(ws, torch.cuda.current_stream())
    # ---- enlarge to B′ = site ⊗ kept ----
    site, lists = blockops.enlarge_right_lists(T, V, mc, left, S, B)
    space2 = d.space_at(bond - 1)                              # bond i−1: A′ | B′
    keys_Bp = blockops.right_block_keys(S + B, left)
    specs_Bp = [blockops.right_operator_spec(k, mc) for k in keys_Bp]
    sp_E = dmrgk.Space(ctx, nc, space2.sectors_B)
    ops_E = DeviceOps(ctx, sp_E, specs_Bp, dev)
    ops_E.arena.fill_(float("nan"))
    index_K = {k: i for i, k in enumerate(keys_B)}
    terms = []
    for o, key in enumerate(keys_Bp):
        for (k, tr, y, odd) in lists[key]:
            terms.append((o, None if k is None else ops_K.ops[index_K[k]], tr, bool(odd), 1.0, blockops.fold_site_parity(site, k, y)))
    enl = dmrgk.Enlarge(ctx, sp_K, sp_E, site.charges, ops_E.ops, terms, site_major=True)
    enl.apply(torch.cuda.current_stream())
    torch.cuda.synchronize()
    YBp = fock_right_set(T, V, mc, len(left))
    for i, key in enumerate(keys_Bp):
        ref = cut_blocks(space2.B.Phi.T @ (YBp[key] @ space2.B.Phi), space2.sectors_B, space2.sectors_B, specs_Bp[i][0])
        got, pad_ok = ops_E.download(i)
        assert pad_ok and set(got) == set(ref), key
        scale = max(1.0, max((np.abs(v).max() for v in ref.values() if v.size), default=1.0))
        err = max((np.abs(got[k] - ref[k]).max() for k in ref if ref[k].size), default=0.0)
        assert err <= 1e-11 * scale, (key, err)
    # ---- σ of bond i−1 with the device-formed R operators (L operators from the oracle) ----
    Heff, P = d.heff_at(space2)
    x = d.guess_at(space2, P)
    ops, tms = [], []
    index_E = {k: i for i, k in enumerate(keys_Bp)}
    for key in keys_Bp:
        dq, par = blockops.right_operator_spec(key, mc)
        ops.append({"half": "B", "dq": dq, "parity": par, "blocks": {}})
    for t in oterms.complementary_terms(T, V, len(left), mc, prune=False):
        fam, lab = t.family, tuple(t.label)
        Rk, tR = {"F1": (("c+",) + lab, False), "F1h": (("c+",) + lab, True), "F2": (("S",) + lab, False),
                  "F2h": (("S",) + lab, True), "F3": (("P",) + lab, False), "F3h": (("P",) + lab, True)}.get(fam, (None, False))
        if fam == "F0":
            Rk = ("H",) if lab == ("B",) else None
        if fam == "F4":
            Rk, tR = (("Q",) + lab, False) if lab[0] <= lab[1] else (("Q", lab[1], lab[0]), True)
        Li = None
        if not (fam == "F0" and lab == ("B",)):
            Xd = space2.A.Phi.T @ (t.X @ space2.A.Phi)
            ops.append({"half": "A", "dq": tuple(t.dq_A), "parity": t.parity,
                        "blocks": cut_blocks(Xd, space2.sectors_A, space2.sectors_A, tuple(t.dq_A))})
            Li = len(ops) - 1
        tms.append((Li, None if Rk is None else index_E[Rk], t.coef, False, tR))
    dp = problem.DeviceProblem(nc, space2.sectors_A, space2.sectors_B, space2.target, ctx=ctx)
    dp.create_ops([(o["half"], o["dq"], o["parity"]) for o in ops])
    dp.alloc_resident()
    for i, o in enumerate(ops):
        if o["half"] == "A":
            dp.set_op_host(i, o["blocks"])
        elif dp.ops[i].n_padded:
            dp.op_views[i].copy_(ops_E.views[i][:dp.ops[i].n_padded])
    dp.build(tms)
    sigma = dp.to_blocks(dp.apply(dp.psi_from_host(dmrg.vec_to_blocks(space2, x))))
    assert rel_max(sigma, dmrg.vec_to_blocks(space2, Heff @ x)) <= TOL_SIGMA
