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
