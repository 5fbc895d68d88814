"""Device-side set-up of one H_eff problem through the C ABI (marshalling and memory only).

``DeviceProblem`` turns plain descriptions — sector lists, stored operators, operator-pair terms —
into library handles and PyTorch-owned device arenas.  Operator values come either from host block
dictionaries (small problems, e.g. a DMRG bond exported by the test-suite) or from the library's
seeded fill kernel (large synthetic workloads of ``workloads``; nothing is shipped from the host).
No arithmetic of the method happens here.
"""
import numpy as np
import torch

from . import dmrgk


def _unpadded_from_blocks(table, blocks):
    """Concatenate host blocks in the library's block-table order."""
    r, c, rows, cols, _, _ = table
    parts = []
    for i in range(len(r)):
        b = np.asarray(blocks[(int(r[i]), int(c[i]))], dtype=np.float64)
        assert b.shape == (rows[i], cols[i]), (b.shape, rows[i], cols[i])
        parts.append(b.reshape(-1))
    return np.concatenate(parts) if parts else np.zeros(0)


def _blocks_from_unpadded(table, u):
    r, c, rows, cols, _, _ = table
    out, o = {}, 0
    for i in range(len(r)):
        n = int(rows[i]) * int(cols[i])
        out[(int(r[i]), int(c[i]))] = u[o:o + n].reshape(int(rows[i]), int(cols[i])).copy()
        o += n
    return out


class DeviceProblem:
    def __init__(self, n_charges, sectors_A, sectors_B, target, device=0, ctx=None):
        if not torch.cuda.is_available():
            raise RuntimeError("dmrgk needs a CUDA device: there is no CPU fallback")
        self.device = torch.device("cuda", device)
        self.ctx = ctx or dmrgk.Ctx(device)
        self.A = dmrgk.Space(self.ctx, n_charges, sectors_A)
        self.B = dmrgk.Space(self.ctx, n_charges, sectors_B)
        self.layout = dmrgk.Layout(self.ctx, self.A, self.B, target)
        self.table = self.layout.blocks()
        self.ops = []
        self.op_arena = None
        self.pinned_arenas = []
        self.pinned_views = {}
        self.heff = None
        self.workspace = None
        self.stream = torch.cuda.current_stream(self.device)
        self.copy_stream = torch.cuda.Stream(self.device)

    # ---- operators ------------------------------------------------------------------------------
    def create_ops(self, specs):
        """specs: [(half, dq, parity)] → handles; one device arena sized for all of them."""
        self.ops = [dmrgk.Op(self.ctx, self.A if half == "A" else self.B, dq, parity)
                    for (half, dq, parity) in specs]
        self.op_offsets = np.concatenate([[0], np.cumsum([op.n_padded for op in self.ops])]).astype(np.int64)
        return self.ops

    def alloc_resident(self, which=None):
        """One arena for the resident operators (all by default); binds them."""
        which = list(range(len(self.ops))) if which is None else list(which)
        sizes = [self.ops[i].n_padded for i in which]
        total = int(sum(sizes))
        self.op_arena = torch.empty(max(total, 16), dtype=torch.float64, device=self.device)
        views, o = {}, 0
        for i, s in zip(which, sizes):
            views[i] = self.op_arena[o:o + s] if s else self.op_arena[0:0]
            if s:
                self.ops[i].bind_device(views[i])
            else:
                self.ops[i].bind_device(self.op_arena[0:16])
            o += s
        self.op_views = views
        return views

    def alloc_pinned(self, which):
        """Pinned host arenas for staged operators; returns {index: pinned tensor}."""
        out = {}
        for i in which:
            t = torch.empty(max(self.ops[i].n_padded, 16), dtype=torch.float64).pin_memory()
            self.ops[i].bind_pinned(t)
            self.pinned_arenas.append(t)
            out[i] = t
        self.pinned_views.update(out)
        return out

    def set_op_host(self, i, blocks):
        """Upload host blocks {(row_idx, col_idx): ndarray} into resident operator i."""
        op = self.ops[i]
        packed = op.pack(_unpadded_from_blocks(op.blocks(), blocks))
        if op.n_padded:
            self.op_views[i].copy_(torch.from_numpy(packed))

    def fill_op(self, i, seed, stream_id, scale_mode, symmetric, arena=None):
        """Seeded values generated on the device (harness kernel, outside the hot path)."""
        op = self.ops[i]
        if op.n_padded:
            op.fill_normal(self.op_views[i] if arena is None else arena, seed, stream_id, scale_mode, symmetric,
                           self.stream)

    def read_op_blocks(self, i, arena=None):
        """D2H of one operator as {(row_idx, col_idx): ndarray} (for CPU references at full size)."""
        op = self.ops[i]
        if not op.n_padded:
            return {}
        src = self.op_views[i] if arena is None else arena
        r, c, rows, cols, ld, off = op.blocks()
        host = src.cpu().numpy()
        out = {}
        for b in range(len(r)):
            n = dmrgk.block_size(rows[b], cols[b])
            out[(int(r[b]), int(c[b]))] = dmrgk.block_unpack(host[off[b]:off[b] + n], rows[b], cols[b])
        return out

    # ---- H_eff ----------------------------------------------------------------------------------
    def build(self, terms, **opts):
        """terms: [(L index or None, R index or None, coef, trans_L, trans_R)]."""
        t = [(None, None, c, "hc", "hc") if tL == "hc" else
             (None if L is None else self.ops[L], None if R is None else self.ops[R], c, tL, tR)
             for (L, R, c, tL, tR) in terms]
        self.heff = dmrgk.Heff(self.ctx, self.layout, t, **opts)
        self.workspace = torch.empty(max(self.heff.workspace_bytes, 128), dtype=torch.uint8, device=self.device)
        return self.heff

    def new_vector(self, zero=True):
        n = max(self.layout.n_padded, 16)
        return (torch.zeros if zero else torch.empty)(n, dtype=torch.float64, device=self.device)

    def psi_from_host(self, blocks):
        packed = self.layout.pack(_unpadded_from_blocks(self.table, blocks))
        v = self.new_vector()
        if self.layout.n_padded:
            v[:self.layout.n_padded].copy_(torch.from_numpy(packed))
        return v

    def psi_fill(self, seed, stream_id):
        v = self.new_vector()
        if self.layout.n_padded:
            self.layout.fill_normal(v, seed, stream_id, self.stream)
        return v

    def to_blocks(self, vec):
        """Packed device vector → {(a_idx, b_idx): ndarray}."""
        if not self.layout.n_padded:
            return {}
        host = vec[:self.layout.n_padded].cpu().numpy()
        return _blocks_from_unpadded(self.table, self.layout.unpack(host))

    def apply(self, psi, sigma=None):
        sigma = self.new_vector(zero=False) if sigma is None else sigma
        self.heff.apply(psi, sigma, self.workspace, self.stream, self.copy_stream)
        return sigma

    def expect(self, psi, n_pairs):
        """⟨ψ, c_k (L_k ⊗ R_k) ψ⟩ for the n_pairs pairs of a plan built with per_pair_output=1 (device tensor)."""
        out = torch.empty(max(n_pairs, 1), dtype=torch.float64, device=self.device)
        self.heff.expect(psi, out, self.workspace, self.stream, self.copy_stream)
        return out[:n_pairs]

    def diag(self, out=None):
        out = self.new_vector(zero=False) if out is None else out
        self.heff.diag(out, self.workspace, self.stream, self.copy_stream)
        return out

    def davidson(self, m_max=16, tol=1e-9, max_iter=500, diag_hook=None):
        """Allocates the basis, the diagonal and the extended workspace; returns a dmrgk.Davidson.
        ``diag_hook`` (k-sharding): applied to the diagonal of this rank's share (the all-reduce)."""
        n = self.layout.n_padded
        self.diag_vec = self.diag()
        if diag_hook is not None:
            diag_hook(self.diag_vec)
        self.V = torch.empty(m_max * n, dtype=torch.float64, device=self.device)
        self.W = torch.empty(m_max * n, dtype=torch.float64, device=self.device)
        wb = (self.heff.workspace_bytes + 127) // 128 * 128
        self.dav_ws = torch.empty(wb + dmrgk.davidson_extra_bytes(m_max, n), dtype=torch.uint8, device=self.device)
        return dmrgk.Davidson(self.heff, m_max, tol, max_iter, self.V, self.W, self.diag_vec, self.dav_ws,
                              self.stream, self.copy_stream)


def from_workload(wl, device=0, pinned=(), ctx=None, **opts):
    """A seeded ``workloads.Workload`` on the device: operators filled by the library's fill kernel
    with the same counter-based stream ids as ``workloads.fill_op_host``."""
    import time
    from workloads import op_stream_of   # input recipe only (no arithmetic of the method)
    t0 = time.perf_counter()
    dp = DeviceProblem(wl.n_charges, wl.sectors_A, wl.sectors_B, wl.target, device, ctx)
    dp.create_ops([(s.half, s.dq, s.parity) for s in wl.ops])
    t1 = time.perf_counter()
    pinned = set(pinned)
    dp.alloc_resident([i for i in range(len(wl.ops)) if i not in pinned])
    staged = dp.alloc_pinned(sorted(pinned))
    for i, s in enumerate(wl.ops):
        mode = 0 if s.scale_mode == "one" else 1
        if i in pinned:
            if dp.ops[i].n_padded:
                tmp = torch.empty(dp.ops[i].n_padded, dtype=torch.float64, device=dp.device)
                dp.fill_op(i, wl.seed, op_stream_of(wl, i), mode, s.symmetric, arena=tmp)
                staged[i][:dp.ops[i].n_padded].copy_(tmp)
        else:
            dp.fill_op(i, wl.seed, op_stream_of(wl, i), mode, s.symmetric)
    torch.cuda.synchronize(dp.device)
    t2 = time.perf_counter()
    dp.build([(t.L, t.R, t.coef, t.trans_L, t.trans_R) for t in wl.terms], **opts)
    t3 = time.perf_counter()
    # "Tables" (Fig. 7) = sector index + operator block tables + task-list build;
    # the seeded fill stands in for the operators a sweep would already hold on the device
    dp.setup_seconds = {"structures": t1 - t0, "fill": t2 - t1, "tasklist": t3 - t2}
    return dp


def from_host(n_charges, sectors_A, sectors_B, target, ops, terms, device=0, ctx=None, **opts):
    """A problem given as host data: ops = [{"half", "dq", "parity", "blocks"}], terms as in build()."""
    dp = DeviceProblem(n_charges, sectors_A, sectors_B, target, device, ctx)
    dp.create_ops([(o["half"], o["dq"], o["parity"]) for o in ops])
    dp.alloc_resident()
    for i, o in enumerate(ops):
        dp.set_op_host(i, o["blocks"])
    dp.build(terms, **opts)
    return dp


class RenormProblem:
    """Device set-up of one renormalisation step (marshalling and memory only): the operators of one
    half of a DeviceProblem as inputs, Φ, and freshly allocated output operators on the kept space."""

    def __init__(self, dp, half, sectors_new, op_indices=None, **opts):
        self.dp, self.ctx, self.device = dp, dp.ctx, dp.device
        self.enl = dp.A if half == "A" else dp.B
        self.kept = dmrgk.Space(self.ctx, self.enl.n_charges, sectors_new)
        self.phi = dmrgk.Iso(self.ctx, self.enl, self.kept)
        self.phi_arena = torch.zeros(max(self.phi.n_padded, 16), dtype=torch.float64, device=self.device)
        self.phi.bind_device(self.phi_arena)
        self.idx = [i for i, op in enumerate(dp.ops) if op.space is self.enl] if op_indices is None else list(op_indices)
        self.ops_in = [dp.ops[i] for i in self.idx]
        self.opts = opts
        self.ops_out, self.out_views, self.plan, self.workspace = [], [], None, None

    def set_phi_host(self, blocks):
        self.phi_arena[:self.phi.n_padded].copy_(torch.from_numpy(self.phi.pack(_unpadded_from_blocks(self.phi.blocks(), blocks))))

    def fill_phi(self, seed, stream_id):
        if self.phi.n_padded:
            self.phi.fill_normal(self.phi_arena, seed, stream_id, self.dp.stream)

    def build(self, specs):
        """specs: [(dq, parity)] of the operators in self.idx order."""
        self.ops_out = [dmrgk.Op(self.ctx, self.kept, dq, parity) for (dq, parity) in specs]
        total = int(sum(op.n_padded for op in self.ops_out))
        self.out_arena = torch.full((max(total, 16),), float("nan"), dtype=torch.float64, device=self.device)
        o = 0
        for op in self.ops_out:
            view = self.out_arena[o:o + op.n_padded] if op.n_padded else self.out_arena[0:16]
            op.bind_device(view)
            self.out_views.append(view)
            o += op.n_padded
        self.plan = dmrgk.Renorm(self.ctx, self.phi, self.ops_in, self.ops_out, **self.opts)
        self.workspace = torch.empty(max(self.plan.workspace_bytes, 128), dtype=torch.uint8, device=self.device)
        return self.plan

    def apply(self):
        self.plan.apply(self.workspace, self.dp.stream)

    def read_out_blocks(self, j):
        """D2H of output operator j as {(row_idx, col_idx): ndarray} plus a flag that its padding is zero."""
        op = self.ops_out[j]
        if not op.n_padded:
            return {}, True
        r, c, rows, cols, ld, off = op.blocks()
        host = self.out_views[j].cpu().numpy()
        out, pad_ok = {}, True
        for b in range(len(r)):
            blk = host[off[b]:off[b] + dmrgk.block_size(rows[b], cols[b])]
            out[(int(r[b]), int(c[b]))] = dmrgk.block_unpack(blk, rows[b], cols[b])
            pad_ok = pad_ok and dmrgk.block_padding_is_zero(blk, rows[b], cols[b])
        return out, pad_ok
