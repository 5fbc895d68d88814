"""The seeded input generators: fixed bits, recipe goldens, term counts."""
import numpy as np

import workloads as w
from _util import golden_table


def test_splitmix64_reference_vector():
    # published SplitMix64 test vector: state 0 → first output 0xE220A8397B1DCDAF
    assert int(w.splitmix64(np.uint64(0))) == 0xE220A8397B1DCDAF


def test_normal12_moments_and_determinism():
    x = w.normal12(1, 2, np.arange(400000))
    assert abs(x.mean()) < 5e-3 and abs(x.var() - 1.0) < 5e-3 and np.abs(x).max() < 6.0
    assert np.array_equal(x[1000:1010], w.normal12(1, 2, np.arange(1000, 1010)))
    assert not np.array_equal(x[:10], w.normal12(1, 3, np.arange(10)))
    # exact dyadic rationals: x·2^32 is an integer
    assert np.all(x * 4294967296.0 == np.round(x * 4294967296.0))


def test_sector_recipes_match_golden():
    g = golden_table("sectors.txt")
    c2 = w.synthetic_config2()
    assert [d for _, d in c2.sectors_A] == [int(v) for v in g["config2"].split()]
    assert c2.M_A == 1024 and len(c2.terms) == 512
    c3 = w.lattice_workload("spinless", 32, 4096, 3)
    dims = [d for _, d in c3.sectors_A]
    head = [int(v) for v in g["config3_head"].split()]
    assert dims[:17] == head and dims == dims[::-1] and sum(dims) == 4096


def test_term_counts_of_the_lattice_workloads():
    # K = 2 + 2n_B + 2n_A + n_A(n_A−1) + n_A²
    assert len(w.lattice_workload("spinless", 32, 4096, 3).terms) == 2146
    c4 = w.lattice_workload("hubbard", 18, 16384, 4)
    assert len(c4.terms) == 2702 and c4.M_A == 16384
    assert sum(1 for _, d in c4.sectors_A if d > 1) == 145
    from collections import Counter
    shifts = Counter()
    for t in c4.terms:
        op = c4.ops[t.L] if t.L is not None else None
        dq = (0, 0) if op is None else tuple(op.dq)
        if t.trans_L:
            dq = tuple(-x for x in dq)
        shifts[dq] += 1
    assert shifts[(0, 0)] == 2 + 2 * 18 * 18 and shifts[(1, 0)] == 36 and shifts[(2, 0)] == 153
    assert shifts[(1, 1)] == 324 and shifts[(1, -1)] == 324 and shifts[(-1, 1)] == 324


def test_config2_shifts_and_blocks():
    c2 = w.synthetic_config2()
    ds = [c2.ops[t.L].dq[0] for t in c2.terms]
    assert set(ds) == {-2, -1, 0, 1, 2}
    for t in c2.terms:
        assert c2.ops[t.L].dq[0] + c2.ops[t.R].dq[0] == 0
        assert c2.ops[t.L].parity == c2.ops[t.R].parity == abs(c2.ops[t.L].dq[0]) % 2
    tab = w.op_block_table(c2.sectors_A, (2,))
    assert len(tab) == 31 and tab[0][:4] == (2, 0, 1, 1)


def test_symmetric_ops_are_symmetric():
    wl = w.lattice_workload("spinless", 5, 24, seed=3)
    i = next(i for i, o in enumerate(wl.ops) if o.symmetric)
    for blk in w.fill_op_host(wl, i).values():
        assert np.array_equal(blk, blk.T)


def test_su2_singlet_workload_structure():
    """The spin-adapted input recipe: multiplet counts against the Fock-space dimension,
    sector labels, one stored operator per Δ(2S), ranks."""
    import workloads as wlmod
    for n in (1, 2, 3, 5):      # Σ (2S+1)·#multiplets = 4^n
        tot = sum((t + 1) * wlmod.su2_multiplet_count(n, N, t) for N in range(2 * n + 1) for t in range(0, n + 1))
        assert tot == 4 ** n
    assert [wlmod.su2_multiplet_count(1, N, t) for (N, t) in ((0, 0), (1, 1), (2, 0), (1, 0), (2, 2))] == [1, 1, 1, 0, 0]
    wl = wlmod.su2_singlet_workload(6, 900, seed=16)
    assert sum(d for _, d in wl.sectors_A) == 900 == sum(d for _, d in wl.sectors_B)
    assert all((N + t) % 2 == 0 and t >= 0 for (N, t), _ in wl.sectors_A)          # N + 2S even: the library's sign never fires
    assert [(N, -t) for (N, t), _ in wl.sectors_A] == [q for q, _ in wl.sectors_B]
    assert len(wl.ranks) == len(wl.terms) == 2 + 4 * 12 + 2 * 66 + 2 * 66 + 12      # the U(1)×U(1) count of 12 spin-orbitals per half
    for t, k2 in zip(wl.terms, wl.ranks):
        if t.L is not None and t.R is not None:
            dl, dr = wl.ops[t.L].dq, wl.ops[t.R].dq
            assert dl[0] == -dr[0] and dl[1] == -dr[1] and abs(dl[1]) <= k2 and (dl[1] - k2) % 2 == 0
    blocks = wlmod.psi_block_table(wl.sectors_A, wl.sectors_B, wl.target)
    assert len(blocks) == len(wl.sectors_A)                                          # every A sector has its singlet partner
