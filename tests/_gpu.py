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
    from paper_2311_14106_b200 import dmrgk
    r, c, rows, cols, ld, off = dp.table
    host = vec[:dp.layout.n_padded].cpu().numpy()
    for b in range(len(r)):
        blk = host[off[b]:off[b] + dmrgk.block_size(rows[b], cols[b])]
        if not dmrgk.block_padding_is_zero(blk, rows[b], cols[b]):
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


# ---- full-size parity: the oracle on sampled output blocks, inputs read back from the device ----
# "the CPU reference at full size reads the *device-generated* blocks back D2H so both
# sides see identical bits".  The device values are the seeded recipe of workloads/ (the harness fill
# kernel is pinned bit-identical to workloads.fill_op_host in test_gpu_heff.py, and `check_inputs`
# below re-checks a sample of the very blocks used here against the host generator), so the oracle's
# inputs are the recipe's, never a result of the hot path.
TOL_BLOCK = 1e-10      # per-block relative max-norm (catches a wrong small block the global norm hides)


def sample_output_blocks(table, n_quantiles=5):
    """≥ 8 sampled ψ/σ blocks: the largest, the smallest (size-1 tail), the
    first and last block of the sector range (edges), and ragged blocks (rows, cols not multiples of
    8 where possible) at area quantiles in between."""
    r, c, rows, cols, _, _ = table
    area = [int(rows[i]) * int(cols[i]) for i in range(len(r))]
    order = sorted(range(len(r)), key=lambda i: area[i])
    picks = [order[-1], order[0], 0, len(r) - 1]
    ragged = lambda i: (rows[i] % 8 != 0) + (cols[i] % 8 != 0)
    for q in range(1, n_quantiles + 1):
        centre = q * (len(order) - 1) // (n_quantiles + 1)
        window = order[max(0, centre - 3):centre + 4]
        picks.append(max(window, key=lambda i: (ragged(i), -abs(order.index(i) - centre))))
    out = []
    for i in picks:
        key = (int(r[i]), int(c[i]))
        if key not in out:
            out.append(key)
    return out


class DeviceInputs:
    """Operator blocks of a DeviceProblem read back D2H one block at a time (resident arenas or the
    pinned host arenas of staged operators)."""

    def __init__(self, wl, dp):
        self.wl, self.dp = wl, dp
        self.tables, self.by_row, self.by_col = {}, {}, {}
        self.n_read = 0
        self.checked = 0

    def table(self, i):
        if i not in self.tables:
            r, c, rows, cols, ld, off = self.dp.ops[i].blocks()
            self.tables[i] = {(int(r[b]), int(c[b])): (int(rows[b]), int(cols[b]), int(ld[b]), int(off[b]))
                              for b in range(len(r))}
            self.by_row[i] = {k[0]: k for k in self.tables[i]}
            self.by_col[i] = {k[1]: k for k in self.tables[i]}
        return self.tables[i]

    def stored_block_with_output(self, i, trans, out):
        """(input sector, stored key) of the block of operator i that, as applied, writes sector `out`."""
        self.table(i)
        key = (self.by_col if trans else self.by_row)[i].get(out)
        if key is None:
            return None, None
        return (key[0] if trans else key[1]), key

    def block(self, i, key):
        from paper_2311_14106_b200 import dmrgk
        rows, cols, ld, off = self.table(i)[key]
        src = self.dp.op_views[i] if i in self.dp.op_views else self.dp.pinned_views[i]
        packed = src[off:off + dmrgk.block_size(rows, cols)].cpu().numpy()
        blk = dmrgk.block_unpack(packed, rows, cols)       # index translation only (panel layout → dense)
        self.n_read += blk.size
        return blk

    def check_inputs(self, i, key, blk, budget=3_000_000):
        """Bit-identity of a read-back block with the seeded host recipe (bounded volume)."""
        import workloads as wlmod
        if self.checked + blk.size > budget:
            return
        ref = wlmod.fill_op_host(self.wl, i, only_blocks={key})[key]
        assert np.array_equal(blk, ref), ("device input differs from the seeded recipe", i, key)
        self.checked += blk.size


def oracle_sigma_on_block(wl, inputs, a_out, b_out, psi_blocks, terms_per_call=96, want_diag=False, coef_of=None):
    """σ[(a_out, b_out)] (and optionally diag(H_eff) on that block) from oracle.heff.sigma_blockwise.

    For every term only the stored L block whose APPLIED output sector is a_out and the R block whose
    applied output sector is b_out can contribute; they are fetched only if the input pair is a ψ
    block.  The term list is cut into groups (k-additivity of the sum) so that host
    memory holds a bounded number of operator blocks at a time; the oracle itself is called unchanged.
    ``coef_of(k, (a_in, b_in))`` supplies the per-(pair, input block) scalar of a spin-adapted problem."""
    from oracle import heff
    psi_keys = set(psi_blocks)
    terms = [(t.L, t.R, t.coef, t.trans_L, t.trans_R) for t in wl.terms]
    sigma, diag = None, None

    def needed(idx, trans, out):
        if idx is None:
            return out, None
        return inputs.stored_block_with_output(idx, trans, out)

    for g0 in range(0, len(terms), terms_per_call):
        ops = [{"half": s.half, "dq": tuple(s.dq), "parity": s.parity, "blocks": {}} for s in wl.ops]
        sub, bc = [], {}
        for k_glob, (L, R, coef, tL, tR) in enumerate(terms[g0:g0 + terms_per_call], start=g0):
            a_in, kl = needed(L, tL, a_out)
            b_in, kr = needed(R, tR, b_out)
            if a_in is None or b_in is None or (a_in, b_in) not in psi_keys:
                continue
            for idx, key in ((L, kl), (R, kr)):
                if idx is not None and key not in ops[idx]["blocks"]:
                    blk = inputs.block(idx, key)
                    inputs.check_inputs(idx, key, blk)
                    ops[idx]["blocks"][key] = blk
            sub.append((L, R, coef, tL, tR))
            if coef_of is not None:
                bc[(len(sub) - 1, (a_in, b_in))] = coef_of(k_glob, (a_in, b_in))
        if not sub:
            continue
        pb = heff.Problem(wl.n_charges, list(wl.sectors_A), list(wl.sectors_B), tuple(wl.target), ops, sub,
                          psi_blocks, wl.name, bc if coef_of is not None else None)
        part = heff.sigma_blockwise(pb)[(a_out, b_out)]
        sigma = part if sigma is None else sigma + part
        if want_diag:
            d = heff.diagonal_blockwise(pb)[(a_out, b_out)]
            diag = d if diag is None else diag + d
    if sigma is None:
        shape = psi_blocks[(a_out, b_out)].shape
        sigma, diag = np.zeros(shape), np.zeros(shape)
    return (sigma, diag) if want_diag else sigma
