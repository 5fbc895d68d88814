"""Test helper: the SU(2)-adapted (spin-singlet) effective Hamiltonian of the two-site Hubbard dimer as a
block-list Problem with per-block-pair scalars.

Each site has three multiplets — |0⟩ (N=0, j=0), the doublet {|↑⟩,|↓⟩} (N=1, j=½), |↑↓⟩ (N=2, j=0) — so the
spin-adapted block dimension is 3 where the U(1)×U(1) one is 4 ("D counts multiplets").  Sectors
are labelled (N, 2j); for the singlet target the right half is labelled (N, −2j) so that the charges of a ψ
block add up to the target (2, 0).  The singlet two-site space has the three states
    |a⟩ = |0; ↑↓⟩ ,   |b⟩ = (c†_{1↑}c†_{2↓} − c†_{1↓}c†_{2↑})/√2 |vac⟩ ,   |c⟩ = |↑↓; 0⟩ ,
and H = −t Σ_σ (c†_{1σ}c_{2σ} + h.c.) + U Σ_i n_{i↑}n_{i↓} restricted to it is
    [[U, −√2 t, 0], [−√2 t, 0, −√2 t], [0, −√2 t, U]]   (up to the phase convention of |b⟩),
lowest eigenvalue (U − √(U² + 16t²))/2 (tests/golden/closed_forms.txt).  The rank-½ operator c† is split
into one stored operator per Δ(2j) = ±1; the stored reduced matrix elements are set to 1 and the product
⟨j′_A‖c†‖j_A⟩⟨j′_B‖c‖j_B⟩ × (recoupling coefficient) × (−t) = −√2 t of each allowed block pair — together with
the compensation of the library's fermionic sign — is what the per-block scalar carries."""
import numpy as np

from oracle.heff import Problem


def dimer_singlet_problem(t=1.0, U=4.0):
    sectors_A = [((0, 0), 1), ((1, 1), 1), ((2, 0), 1)]
    sectors_B = [((0, 0), 1), ((1, -1), 1), ((2, 0), 1)]
    one = np.ones((1, 1))
    ops = [
        {"half": "A", "dq": (1, 1), "parity": 1, "blocks": {(1, 0): one}},        # 0: c† : (0,0) → (1,1)
        {"half": "A", "dq": (1, -1), "parity": 1, "blocks": {(2, 1): one}},       # 1: c† : (1,1) → (2,0)
        {"half": "B", "dq": (-1, -1), "parity": 1, "blocks": {(1, 2): one}},      # 2: c  : (2,0) → (1,−1)
        {"half": "B", "dq": (-1, 1), "parity": 1, "blocks": {(0, 1): one}},       # 3: c  : (1,−1) → (0,0)
        {"half": "A", "dq": (0, 0), "parity": 0, "blocks": {(0, 0): 0 * one, (1, 1): 0 * one, (2, 2): U * one}},   # 4: H_A
        {"half": "B", "dq": (0, 0), "parity": 0, "blocks": {(0, 0): 0 * one, (1, 1): 0 * one, (2, 2): U * one}},   # 5: H_B
    ]
    # ψ blocks in A order: (0|2) = (a=0,b=2), (1|1) = (1,1), (2|0) = (2,0)
    terms = [(0, 2, -t, False, False),      # a → b
             (1, 3, -t, False, False),      # b → c
             (0, 2, -t, True, True),        # b → a
             (1, 3, -t, True, True),        # c → b
             (4, None, 1.0, False, False), (None, 5, 1.0, False, False)]
    r2 = np.sqrt(2.0)
    # In the (N, 2j) labelling N + 2j is even for every sector (N odd ⇔ j half-integer), so the library's
    # fermionic sign (−1)^{π·Σ charges of the input A sector} never fires: the whole phase of a block pair,
    # Jordan–Wigner sign included, is carried by the per-block scalar.
    block_coef = {(0, (0, 2)): r2, (1, (1, 1)): r2, (2, (1, 1)): r2, (3, (2, 0)): r2}
    psi = {(0, 2): np.array([[0.3]]), (1, 1): np.array([[-0.5]]), (2, 0): np.array([[0.8]])}
    H = np.array([[U, -r2 * t, 0.0], [-r2 * t, 0.0, -r2 * t], [0.0, -r2 * t, U]])
    return Problem(2, sectors_A, sectors_B, (2, 0), ops, terms, psi, "dimer_su2", block_coef), H
