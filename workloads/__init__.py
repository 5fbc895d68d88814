"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This package holds *inputs only*: a counter-based random stream, the sector-size
recipe and the operator-pair lists (charge shifts, parities, coefficients,
transpose pairing) of the five BASELINE.json workloads.  It contains none of
the method's arithmetic (no product, no sign rule, no accumulation) and imports
neither ``oracle`` nor ``paper_2311_14106_b200``.
"""
from .rng import splitmix64, normal12, uniform_u64, stream_base  # noqa: F401
from .sectors import gaussian_sectors, binom  # noqa: F401
from .configs import (  # noqa: F401
    Workload, OpSpec, TermSpec, synthetic_config2, lattice_workload,
    spinless_term_structure, hubbard_term_structure, op_block_table,
    psi_block_table, fill_op_host, fill_psi_host, op_stream_id, op_stream_of, sub_workload, PSI_STREAM,
    config3, config4, config4_realspace, config5, config5_keep, config5_staged_ops,
    renorm_basis, fill_phi_host, PHI_STREAM, su2_singlet_workload, su2_multiplet_count,
)
