"""-m gpu parity of the renormalisation step O′ = Φᵀ O Φ through the C ABI
against oracle/renorm.py, element by element on the same seeded inputs (1e-11 relative max-norm)."""
import numpy as np
import pytest

import workloads as wlmod
from oracle import renorm, lattice, dmrg, export, terms as terms_mod
from _gpu import rel_max, TOL_SIGMA

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _device(wl, M_new, **opts):
    from paper_2311_14106_b200 import problem
    dp = problem.from_workload(wl)
    sectors_new, table = wlmod.renorm_basis(wl, M_new=M_new)
    rp = problem.RenormProblem(dp, "A", sectors_new, **opts)
    rp.fill_phi(wl.seed, wlmod.PHI_STREAM)
    rp.build([(wl.ops[i].dq, wl.ops[i].parity) for i in rp.idx])
    return dp, rp, sectors_new, table


def _check_ops(wl, rp, sectors_new, phi, which):
    for j in which:
        i = rp.idx[j]
        op = {"half": "A", "dq": tuple(wl.ops[i].dq), "parity": wl.ops[i].parity, "blocks": wlmod.fill_op_host(wl, i)}
        ref = renorm.renormalise_blockwise(op, wl.sectors_A, phi, sectors_new)
        got, pad_ok = rp.read_out_blocks(j)
        assert pad_ok and set(got) == set(ref), (j, sorted(set(got) ^ set(ref))[:4])
        assert rel_max(got, ref) <= TOL_SIGMA, (j, rel_max(got, ref))


@pytest.mark.parametrize("kernel", [0, 1])
def test_small_all_operators(kernel):
    from paper_2311_14106_b200 import dmrgk
    wl = wlmod.lattice_workload("spinless", 5, 24, seed=3)
    dp, rp, sectors_new, table = _device(wl, 11, kernel=kernel)
    phi = wlmod.fill_phi_host(wl, table)
    # the library's Φ fill reproduces the host generator bit for bit
    r, c, rows, cols, ld, off = rp.phi.blocks()
    host = rp.phi_arena.cpu().numpy()
    for b in range(len(r)):
        packed = host[off[b]:off[b] + dmrgk.block_size(rows[b], cols[b])]
        assert np.array_equal(dmrgk.block_unpack(packed, rows[b], cols[b]), phi[(int(r[b]), int(c[b]))])
        assert dmrgk.block_padding_is_zero(packed, rows[b], cols[b])
    rp.apply()
    torch.cuda.synchronize()
    _check_ops(wl, rp, sectors_new, phi, range(len(rp.idx)))
    assert rp.plan.flops == sum(renorm.flops({"blocks": wlmod.fill_op_host(wl, i)}, phi) for i in rp.idx)


@pytest.mark.parametrize("make,M_new,opts", [
    (lambda: wlmod.lattice_workload("spinless", 10, 600, seed=13, width2=4.0, keep=lambda f, i: f in ("F1", "F2") or i % 5 == 0), 300, {}),
    (lambda: wlmod.lattice_workload("hubbard", 5, 400, seed=14, keep=lambda f, i: f in ("F1", "F2") or i % 7 == 0), 100, {}),
    (lambda: wlmod.lattice_workload("spinless", 10, 600, seed=13, width2=4.0, keep=lambda f, i: f in ("F1", "F2") or i % 5 == 0), 300,
     {"t_chunk_bytes": 1 << 20}),
])
def test_medium_several_tiles_ragged_tails_and_chunks(make, M_new, opts):
    wl = make()
    dp, rp, sectors_new, table = _device(wl, M_new, **opts)
    phi = wlmod.fill_phi_host(wl, table)
    rp.apply()
    rp.apply()          # a second call overwrites with the same values
    torch.cuda.synchronize()
    _check_ops(wl, rp, sectors_new, phi, range(0, len(rp.idx), 3))
    if opts:
        assert rp.plan.n_launches > 2


def test_dmrg_bond_physics():
    """3×3 spinless torus: the exported L_k of a bond, carried by that bond's SVD basis on the GPU,
    equal Φ_new† X_k Φ_new from the Fock-space matrices (the oracle's physics pin, on the device)."""
    from paper_2311_14106_b200 import problem
    T, V, mc = lattice.spinless_tV(3)
    d = dmrg.SimpleDMRG(T, V, mc, [[i] for i in range(9)], (4,), D=6, seed=5)
    d.warmup_to(3)
    space = d.space_at(3)
    pb = export.export_bond(d, space, use_transpose_pairs=False, identity_as_none=False)
    tms = terms_mod.complementary_terms(d.T, d.V, space.A.n_modes, d.mc)
    PhiA = space.A.Phi
    d.step(3, +1)
    new, sectors_new = dmrg.sector_major(d.L[4])
    U = PhiA.T @ new.Phi
    idx_enl = {q: i for i, (q, _) in enumerate(space.sectors_A)}
    sl_e, sl_n = dmrg.sector_slices(space.sectors_A), dmrg.sector_slices(sectors_new)
    phi = {(idx_enl[q], ni): U[sl_e[idx_enl[q]], sl_n[ni]].copy() for ni, (q, _) in enumerate(sectors_new)}
    dp = problem.from_host(pb.n_charges, pb.sectors_A, pb.sectors_B, pb.target, pb.ops, pb.terms)
    rp = problem.RenormProblem(dp, "A", sectors_new)
    rp.set_phi_host(phi)
    a_idx = [i for i, o in enumerate(pb.ops) if o["half"] == "A"]
    assert rp.idx == a_idx and len(a_idx) == len(tms)
    rp.build([(pb.ops[i]["dq"], pb.ops[i]["parity"]) for i in a_idx])
    rp.apply()
    torch.cuda.synchronize()
    off_n = np.concatenate([[0], np.cumsum([dn for _, dn in sectors_new])])
    worst, scale = 0.0, 0.0
    for j, t in enumerate(tms):
        direct = new.Phi.T @ (t.X @ new.Phi)
        scale = max(scale, np.abs(direct).max())
        got, pad_ok = rp.read_out_blocks(j)
        assert pad_ok
        dense = np.zeros_like(direct)
        for (rn, cn), blk in got.items():
            dense[off_n[rn]:off_n[rn] + blk.shape[0], off_n[cn]:off_n[cn] + blk.shape[1]] = blk
        worst = max(worst, np.abs(dense - direct).max())
    assert worst <= 1e-11 * scale


def test_errors():
    from paper_2311_14106_b200 import dmrgk, problem
    wl = wlmod.lattice_workload("spinless", 5, 24, seed=3)
    dp = problem.from_workload(wl)
    sectors_new, _ = wlmod.renorm_basis(wl, M_new=11)
    rp = problem.RenormProblem(dp, "A", sectors_new)
    specs = [(wl.ops[i].dq, wl.ops[i].parity) for i in rp.idx]
    bad = list(specs)
    bad[1] = ((specs[1][0][0] + 1,), specs[1][1])
    with pytest.raises(dmrgk.DmrgkError) as e:
        rp.build(bad)
    assert e.value.status == dmrgk.ECHARGE
    other = problem.RenormProblem(dp, "A", sectors_new)
    other.build(specs)
    with pytest.raises(dmrgk.DmrgkError) as e:          # outputs on a different (equal-looking) kept space
        dmrgk.Renorm(dp.ctx, rp.phi, rp.ops_in, other.ops_out)
    assert e.value.status == dmrgk.ESHAPE
    unbound = [dmrgk.Op(dp.ctx, rp.kept, dq, par) for dq, par in specs]
    with pytest.raises(dmrgk.DmrgkError) as e:
        dmrgk.Renorm(dp.ctx, rp.phi, rp.ops_in, unbound)
    assert e.value.status == dmrgk.ESTATE
    too_many = [(q, d + 1) for q, d in wl.sectors_A]    # a kept sector larger than its enlarged sector
    with pytest.raises(dmrgk.DmrgkError) as e:
        problem.RenormProblem(dp, "A", too_many)
    assert e.value.status == dmrgk.ESHAPE
    orphan = list(sectors_new) + [((99,), 2)]           # a kept sector with no enlarged counterpart
    with pytest.raises(dmrgk.DmrgkError) as e:
        problem.RenormProblem(dp, "A", orphan)
    assert e.value.status == dmrgk.ESHAPE and "no enlarged sector" in e.value.message


def test_config4_half_sampled_operators():
    """All 1369 enlarged-block operators of the config-4 left half (≈ 52 GB) renormalised to
    D = 4096 kept states; sampled operators against the oracle (host-generated blocks)."""
    wl = wlmod.config4()
    dp, rp, sectors_new, table = _device(wl, None)
    assert sum(d for _, d in sectors_new) == 4096
    phi = wlmod.fill_phi_host(wl, table)
    rp.apply()
    torch.cuda.synchronize()
    n = len(rp.idx)
    _check_ops(wl, rp, sectors_new, phi, [0, n // 3, n - 1])
