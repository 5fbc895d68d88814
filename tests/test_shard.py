"""k-sharding of the operator-pair list over GPUs on
CPU: the partitioner's invariants, and — with two gloo processes — that the all-reduced sum of the
shards' σ (each shard computed by the ORACLE from its own sub-workload) equals the σ of the full list."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

import workloads as wlmod
from oracle import heff

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _workload():
    thin = lambda fam, i: fam in ("F1", "F2") or i % 2 == 0
    return wlmod.lattice_workload("hubbard", 3, 60, seed=4, keep=thin)


@pytest.mark.parametrize("n_shards", [2, 3, 8])
def test_partition_covers_balances_and_keeps_partners_together(n_shards):
    from paper_2311_14106_b200 import shard
    wl = _workload()
    shards, stats = shard.partition_pairs(wl, n_shards)
    assert sorted(k for s in shards for k in s) == list(range(len(wl.terms)))      # a partition
    owner = {k: g for g, s in enumerate(shards) for k in s}
    for k, t in enumerate(wl.terms):                                                # h.c. partners share a rank
        for k2, t2 in enumerate(wl.terms):
            if (t.L, t.R) == (t2.L, t2.R):
                assert owner[k] == owner[k2]
    flops, _ = shard.term_costs(wl)
    assert flops.sum() == heff.flops_alg(heff.problem_from_workload(wl, with_psi=False))   # the library's count
    loads = np.array([st["flops"] for st in stats])
    assert loads.sum() == pytest.approx(flops.sum())
    biggest_group = max(flops[[k for k, t in enumerate(wl.terms) if (t.L, t.R) == key]].sum()
                        for key in {(t.L, t.R) for t in wl.terms})
    assert loads.max() - loads.min() <= 2 * biggest_group                           # LPT balance bound
    # no stored operator is held by two ranks
    ops_of = [{i for k in s for i in (wl.terms[k].L, wl.terms[k].R) if i is not None} for s in shards]
    for a in range(n_shards):
        for b in range(a + 1, n_shards):
            assert not (ops_of[a] & ops_of[b])


def test_sub_workload_keeps_operator_values():
    wl = _workload()
    ids = list(range(3, len(wl.terms), 4))
    sub = wlmod.sub_workload(wl, ids)
    used = sorted({i for k in ids for i in (wl.terms[k].L, wl.terms[k].R) if i is not None})
    assert len(sub.ops) == len(used) < len(wl.ops)
    for new, old in enumerate(used):
        a, b = wlmod.fill_op_host(sub, new), wlmod.fill_op_host(wl, old)
        assert set(a) == set(b) and all(np.array_equal(a[k], b[k]) for k in a)


WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r}); sys.path.insert(0, os.path.join({root!r}, "tests"))
import numpy as np, torch, torch.distributed as dist
import workloads as wlmod
from oracle import heff
from paper_2311_14106_b200 import shard
from test_shard import _workload
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank, world = dist.get_rank(), dist.get_world_size()
wl = _workload()
shards, _ = shard.partition_pairs(wl, world)
pb = heff.problem_from_workload(wlmod.sub_workload(wl, shards[rank]))
part = heff.psi_to_vec(pb, heff.sigma_blockwise(pb))          # this rank's partial σ (oracle)
t = torch.from_numpy(part.copy())
dist.all_reduce(t, op=dist.ReduceOp.SUM)                       # what ShardedProblem.allreduce does over NCCL
full = heff.problem_from_workload(wl)
ref = heff.psi_to_vec(full, heff.sigma_blockwise(full))
err = float(np.abs(t.numpy() - ref).max() / np.abs(ref).max())
print(json.dumps({{"rank": rank, "err": err, "n_terms": len(shards[rank]), "partial_norm": float(np.linalg.norm(part))}}), flush=True)
dist.destroy_process_group()
"""


def test_sum_of_shard_sigmas_is_sigma_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = str(s.getsockname()[1])
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=port)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, _ = p.communicate(timeout=300)
        assert p.returncode == 0
        outs.append(json.loads(out.strip().splitlines()[-1]))
    assert sum(o["n_terms"] for o in outs) == len(_workload().terms)
    for o in outs:
        assert o["err"] <= 1e-13 and o["partial_norm"] > 0


@pytest.mark.gpu
def test_shards_applied_one_after_the_other_and_davidson_hook():
    """One GPU: the shards of a two-way split, applied in turn and summed, give the unsharded σ; the
    Davidson driver with the all-reduce hook (here: 'add the other rank's share') reproduces the
    unsharded Ritz values."""
    torch = pytest.importorskip("torch")
    from paper_2311_14106_b200 import problem, shard
    wl = _workload()
    full = problem.from_workload(wl)
    psi = full.psi_fill(wl.seed, wlmod.PSI_STREAM)
    ref = full.apply(psi).clone()
    parts = [shard.ShardedProblem(wl, r, 2) for r in range(2)]
    for sp in parts:
        sp.world = 1                                   # no process group here: the sum is done by hand below
    total = sum(sp.dp.apply(psi).clone() for sp in parts)
    assert float((total - ref).abs().max() / ref.abs().max()) <= 1e-13
    dav_ref = full.davidson(m_max=8, tol=1e-9, max_iter=400)
    dav_ref.start(psi)
    th_ref = dav_ref.solve(None)[0]
    me, other = parts
    dav = me.dp.davidson(m_max=8, tol=1e-9, max_iter=400, diag_hook=lambda d: d.add_(other.dp.diag()))

    def hook(ptr, n):
        W = me.dp.W
        j = (ptr - W.data_ptr()) // (8 * n)
        W[j * n:(j + 1) * n].add_(other.dp.apply(me.dp.V[j * n:(j + 1) * n]))
        return 0

    dav.set_allreduce(hook)
    dav.start(psi)
    theta, rn, n_apply, ok = dav.solve(None)
    assert ok and abs(theta - th_ref) <= 1e-9 * max(1.0, abs(th_ref))
    # the same two results against the oracle (not only CUDA against CUDA): the summed σ against the
    # per-task NumPy products of the full pair list, θ against the lowest eigenvalue of the dense H_eff
    from _gpu import rel_max, TOL_SIGMA
    prob = heff.problem_from_workload(wl)              # ψ from the host recipe (the device fill is pinned to it)
    assert rel_max(full.to_blocks(total), heff.sigma_blockwise(prob)) <= TOL_SIGMA
    H = heff.dense_heff(prob)
    e0 = np.linalg.eigvalsh(H)[0]
    assert abs(theta - e0) <= 1e-9 * max(1.0, abs(e0))


@pytest.mark.gpu
def test_allreduce_hook_runs_on_the_solver_stream_and_reports_failures():
    """The hook's work must be ordered on the solver's main stream even when the caller has made another
    stream current in the meantime (an NCCL all-reduce issued on the wrong stream would read W before the
    apply has written it); a hook that raises, or returns non-zero, stops the driver with ESTATE."""
    torch = pytest.importorskip("torch")
    from paper_2311_14106_b200 import dmrgk, problem, shard
    wl = _workload()
    full = problem.from_workload(wl)
    psi = full.psi_fill(wl.seed, wlmod.PSI_STREAM)
    dav_ref = full.davidson(m_max=8, tol=1e-9, max_iter=400)
    dav_ref.start(psi)
    th_ref = dav_ref.solve(None)[0]
    parts = [shard.ShardedProblem(wl, r, 2) for r in range(2)]
    me, other = parts
    dav = me.dp.davidson(m_max=8, tol=1e-9, max_iter=400, diag_hook=lambda d: d.add_(other.dp.diag()))
    seen = []

    def hook(ptr, n):
        seen.append(torch.cuda.current_stream().cuda_stream)
        W = me.dp.W
        j = (ptr - W.data_ptr()) // (8 * n)
        W[j * n:(j + 1) * n].add_(other.dp.apply(me.dp.V[j * n:(j + 1) * n]))
        return 0

    dav.set_allreduce(hook)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):                      # a foreign current stream while the driver runs
        assert torch.cuda.current_stream().cuda_stream != me.dp.stream.cuda_stream
        dav.start(psi)
        theta, rn, n_apply, ok = dav.solve(None)
    assert ok and abs(theta - th_ref) <= 1e-9 * max(1.0, abs(th_ref))
    assert seen and all(s == me.dp.stream.cuda_stream for s in seen)

    def bad(ptr, n):
        raise RuntimeError("boom")

    for fn in (bad, lambda ptr, n: 3):
        dav.set_allreduce(fn)
        with pytest.raises(dmrgk.DmrgkError) as e:
            dav.start(psi)
        assert e.value.status == dmrgk.ESTATE
