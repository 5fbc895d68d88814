"""k-sharding of the operator-pair list over G GPUs ("new kernel
utilizing … D2D NVLINK"): the sum over pairs is a sum of independent contributions,

    σ = Σ_g σ_g ,   σ_g = Σ_{k ∈ shard g} c_k (L_k ⊗ R_k) ψ ,

so every rank holds only the operators of its shard (G GPUs hold G × 180 GB of operators), ψ is
replicated, each rank applies its shard and ONE all-reduce (sum) of a ψ-sized buffer per matvec makes σ
identical on all ranks; the Davidson iteration then runs replicated and unchanged.

Host logic only (index bookkeeping and a partition heuristic); the products run in the library's
kernels, the all-reduce in NCCL over NVLink (torch.distributed).  No hardware with more than one GPU
was available to this build: the path is covered by CPU tests (gloo, world size 2) and by a one-GPU
test that applies the shards one after the other; its scaling is UNMEASURED.
"""
import numpy as np


def term_costs(wl):
    """Per operator pair: (algorithmic flops of its tasks, bytes of its stored operator blocks).

    flops = Σ over ψ blocks (a, b) whose applied L and R blocks exist of
    min(2m′n(m+n′), 2mn′(n+m′)) (an identity factor leaves one product) — the count
    dmrgk_heff_query reports, here from the sector tables alone."""
    idxA = {q: i for i, (q, _) in enumerate(wl.sectors_A)}
    idxB = {q: i for i, (q, _) in enumerate(wl.sectors_B)}
    dA = [d for _, d in wl.sectors_A]
    dB = [d for _, d in wl.sectors_B]
    blocks = []
    for ai, (qa, da) in enumerate(wl.sectors_A):
        qb = tuple(t - x for t, x in zip(wl.target, qa))
        bi = idxB.get(qb)
        if bi is not None and da > 0 and dB[bi] > 0:
            blocks.append((ai, bi, qa, qb))
    flops = np.zeros(len(wl.terms))
    nbytes = np.zeros(len(wl.terms))
    for k, t in enumerate(wl.terms):
        dl = None if t.L is None else tuple((-x if t.trans_L else x) for x in wl.ops[t.L].dq)
        dr = None if t.R is None else tuple((-x if t.trans_R else x) for x in wl.ops[t.R].dq)
        f = b = 0.0
        for (ai, bi, qa, qb) in blocks:
            ao = ai if dl is None else idxA.get(tuple(x + y for x, y in zip(qa, dl)))
            bo = bi if dr is None else idxB.get(tuple(x + y for x, y in zip(qb, dr)))
            if ao is None or bo is None or dA[ao] == 0 or dB[bo] == 0:
                continue
            m, n, mo, no = dA[ai], dB[bi], dA[ao], dB[bo]
            if dl is None and dr is None:
                continue
            if dl is None:
                f += 2.0 * m * n * no
            elif dr is None:
                f += 2.0 * mo * m * n
            else:
                f += min(2.0 * mo * n * (m + no), 2.0 * m * no * (n + mo))
            if dl is not None:
                b += 8.0 * mo * m
            if dr is not None:
                b += 8.0 * no * n
        flops[k], nbytes[k] = f, b
    return flops, nbytes


def partition_pairs(wl, n_shards, byte_weight=0.25):
    """Split the pair list into ``n_shards`` lists of term indices, balanced by flops and bytes.

    Pairs that share stored operators (a pair and its h.c. partner re-use the same blocks through the
    transpose flags) stay together so that no operator is stored twice.  Groups are assigned longest
    first to the shard with the smallest load, load = flops share + byte_weight · byte share
    (flops decide the matvec time, bytes the HBM footprint).  Deterministic."""
    flops, nbytes = term_costs(wl)
    groups = {}
    for k, t in enumerate(wl.terms):
        groups.setdefault((t.L, t.R), []).append(k)
    items = []
    for key, ks in groups.items():
        items.append((float(flops[ks].sum()), float(nbytes[ks].max()), ks))     # blocks stored once per group
    tf = max(sum(i[0] for i in items), 1.0)
    tb = max(sum(i[1] for i in items), 1.0)
    items.sort(key=lambda i: (-(i[0] / tf + byte_weight * i[1] / tb), i[2][0]))
    load = [0.0] * n_shards
    shards = [[] for _ in range(n_shards)]
    stats = [{"flops": 0.0, "bytes": 0.0} for _ in range(n_shards)]
    for f, b, ks in items:
        g = min(range(n_shards), key=lambda j: (load[j], j))
        shards[g].extend(ks)
        load[g] += f / tf + byte_weight * b / tb
        stats[g]["flops"] += f
        stats[g]["bytes"] += b
    for s in shards:
        s.sort()
    return shards, stats


class ShardedProblem:
    """One rank's share of a k-sharded H_eff: a DeviceProblem over ``sub_workload(wl, shard)`` plus the
    all-reduce that completes σ.  ``group`` is a torch.distributed process group (None = default)."""

    def __init__(self, wl, rank, world, device=0, group=None, **opts):
        import workloads as wlmod
        from . import problem
        self.rank, self.world, self.group = rank, world, group
        self.shards, self.stats = partition_pairs(wl, world)
        self.wl = wlmod.sub_workload(wl, self.shards[rank], name=f"{wl.name}_shard{rank}of{world}")
        self.dp = problem.from_workload(self.wl, device=device, **opts)

    def allreduce(self, sigma):
        if self.world > 1:
            import torch.distributed as dist
            dist.all_reduce(sigma, op=dist.ReduceOp.SUM, group=self.group)
        return sigma

    def apply(self, psi, sigma=None):
        """σ = Σ_g σ_g: local shard apply, then the all-reduce over the ranks."""
        return self.allreduce(self.dp.apply(psi, sigma))

    def davidson(self, **kw):
        """The library's Davidson driver with the all-reduce hooked in after every apply (and after the
        diagonal): every rank iterates on identical data."""
        dav = self.dp.davidson(diag_hook=self.allreduce, **kw)
        dav.set_allreduce(self._reduce_ptr)
        return dav

    def _reduce_ptr(self, ptr, n):
        W, V = self.dp.W, self.dp.V
        for base in (W, V):
            off = ptr - base.data_ptr()
            if 0 <= off < base.numel() * 8:
                self.allreduce(base[off // 8: off // 8 + n])
                return 0
        return -1
