"""CPU oracle for the H_eff·ψ / Davidson hot path of arXiv 2311.14106.

TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct NumPy/SciPy code in
fp64, written from the paper (``/root/reference/PAPER.md``) and the readings
listed in DESIGN.md.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import it.  It
shares no code with the CUDA library (``paper_2311_14106_b200``) and never
imports it; only the seeded input generators in ``workloads/`` serve both.

Tiers:
  T0  fock.py      Jordan-Wigner Fock-space matrices, Eq. (1)-(3) Hamiltonians, ED
      lattice.py   torus bond lists, t/V tensors, mode rotation
  T1  dmrg.py      simple two-site DMRG with explicit block bases; H_eff = P†HP
      terms.py     complementary-operator regrouping of Eq. (1) across a cut
  T2  heff.py      dense Kronecker H_eff = Σ c_k (L_k P^π) ⊗ R_k from block lists
  T3  heff.py      the same sum block by block (one dense product per step);
                   also the timed CPU baseline
      davidson.py  the Davidson iteration, step by step
      renorm.py    renormalisation O′ = Φ† O Φ of block operators

Parity pins: every function here is pinned by ``tests/test_oracle_*.py``
(anticommutators, brute-force bit-string action, free-fermion closed forms,
the Hubbard dimer, spectrum invariance under mode rotation,
‖H − Σ_k c_k (X_k P^π)⊗Y_k‖ on small mode counts, P†HP against the exported
blocks, exact diagonalisation against DMRG at untruncated D).  The paper prints
no σ, no H_eff spectrum and no small-lattice energy, so no value here is pinned
*by the paper's numbers*: "parity unpinned by the paper; pinned by definition +
brute force".
"""
