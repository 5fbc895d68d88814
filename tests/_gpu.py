"""Helpers of the -m gpu parity tests: oracle Problem ↔ device problem, comparisons."""
import functools

import numpy as np

TOL_SIGMA = 1e-11      # BASELINE.json north_star: relative max-norm of σ (reading r12)
TOL_ENERGY = 1e-9      # BASELINE.json north_star: Davidson energies (reading r13)


def device_problem(pb, **opts):
    """oracle.heff.Problem (host block lists) → paper_2311_14106_b200.problem.DeviceProblem."""
    from paper_2311_14106_b200 import problem
    return problem.from_host(pb.n_charges, pb.sectors_A, pb.sectors_B, pb.target, pb.ops, pb.terms, **opts)


def rel_max(got, ref):
    """max_i |got − ref| / max_i |ref| over all stored elements of a block dictionary (r12)."""
    assert set(got) == set(ref)
    num = max((np.abs(got[k] - ref[k]).max() for k in ref if ref[k].size), default=0.0)
    den = max((np.abs(ref[k]).max() for k in ref if ref[k].size), default=0.0)
    return num / den if den > 0 else num


def padding_is_zero(dp, vec):
    """Every padding column of the packed arena must hold exact zeros."""
    r, c, rows, cols, ld, off = dp.table
    host = vec[:dp.layout.n_padded].cpu().numpy()
    for b in range(len(r)):
        blk = host[off[b]:off[b] + int(rows[b]) * int(ld[b])].reshape(int(rows[b]), int(ld[b]))
        if np.any(blk[:, cols[b]:] != 0.0):
            return False
    return True


@functools.lru_cache(maxsize=1)
def config1_problem():
    """BASELINE.json configs[0]: 4×4 spinless torus (t=1, t'=0.4, V=0.8, N=8), snake order, D=64,
    bond "sites 8|9" (1-based) after one warm-up sweep; returns (Problem with ψ, P†HP, x, space)."""
    from oracle import lattice, dmrg, export
    T, V, mc = lattice.spinless_tV(4)
    d = dmrg.SimpleDMRG(T, V, mc, [[i] for i in range(16)], (8,), D=64, seed=1)
    d.warmup_to(7)
    space = d.space_at(7)
    Heff, P = d.heff_at(space)
    x = d.guess_at(space, P)
    pb = export.export_bond(d, space)
    pb.psi = dmrg.vec_to_blocks(space, x)
    return pb, Heff, x, space


def oracle_problem_for_output_block(wl, a_out, b_out, psi=None):
    """oracle.heff.Problem restricted to the operator blocks that write σ block (a_out, b_out) of a
    (large) seeded workload: for every term only the L block whose applied output sector is a_out and
    the R block whose applied output sector is b_out are generated (host generator, workloads.fill_op_host),
    so `sigma_blockwise` of the restricted problem equals the full σ on that block and is zero elsewhere."""
    import workloads as wlmod
    from oracle import heff
    need = {}
    for t in wl.terms:
        for idx, trans, out in ((t.L, t.trans_L, a_out), (t.R, t.trans_R, b_out)):
            if idx is None:
                continue
            spec = wl.ops[idx]
            for (r, c, _, _, _) in wlmod.op_block_table(wl.sectors(spec.half), spec.dq):
                if (c if trans else r) == out:
                    need.setdefault(idx, set()).add((r, c))
    ops = []
    for i, spec in enumerate(wl.ops):
        blocks = wlmod.fill_op_host(wl, i, only_blocks=need[i]) if i in need else {}
        ops.append({"half": spec.half, "dq": tuple(spec.dq), "parity": spec.parity, "blocks": blocks})
    terms = [(t.L, t.R, t.coef, t.trans_L, t.trans_R) for t in wl.terms]
    return heff.Problem(wl.n_charges, list(wl.sectors_A), list(wl.sectors_B), tuple(wl.target), ops, terms,
                        wlmod.fill_psi_host(wl) if psi is None else psi, wl.name + f"_out{a_out}_{b_out}")
