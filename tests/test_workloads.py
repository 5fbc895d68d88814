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
