"""Host logic of paper_2311_14106_b200/su2.py (no GPU): the closed-form singlet recoupling scalar and the
block-coefficient table against the oracle's brute-force Clebsch–Gordan sums."""
import numpy as np
import pytest

from oracle import su2 as osu2, lattice
from paper_2311_14106_b200 import su2


def test_recoupling_closed_form_vs_brute_force_cg_sums():
    for two_s in range(0, 7):
        for two_k in (0, 1, 2, 3, 4):
            for d in range(-two_k, two_k + 1, 2):
                two_s2 = two_s + d
                if two_s2 < 0:
                    assert su2.singlet_recoupling(two_s, two_s2, two_k) == 0.0
                    continue
                want = osu2.recoupling_singlet(two_s, two_s2, two_k)
                assert abs(su2.singlet_recoupling(two_s, two_s2, two_k) - want) < 1e-13, (two_s, two_s2, two_k)
    assert su2.singlet_recoupling(0, 0, 2) == 0.0 and abs(osu2.recoupling_singlet(0, 0, 2)) < 1e-15    # triangle rule
    assert not su2.triangle(1, 1, 1) and su2.triangle(1, 1, 2) and su2.triangle(3, 2, 1)


def test_block_coef_table_vs_oracle_on_a_hubbard_torus():
    from test_oracle_su2 import hubbard
    T, V, mc = hubbard(2, 2, True)
    pb, *_ = osu2.reduced_problem(T, V, 2, 4)
    psi_blocks = pb.psi_blocks()
    meta = []
    for (L, R, c, _, _), k2 in zip(pb.terms, pb.ranks):
        meta.append((0, 0, 0) if L is None or R is None else (k2, pb.ops[L]["parity"], pb.ops[L]["dq"][1]))
    table = su2.block_coef_table(pb.sectors_A, [a for a, _ in psi_blocks], meta)
    seen = 0
    for (k, blk), v in pb.block_coef.items():
        j = psi_blocks.index(blk)
        assert abs(table[k, j] - v) < 1e-13
        seen += 1
    assert seen > 50 and np.any(table < 0) and np.any(np.abs(np.abs(table) - 1.0) > 0.1)
