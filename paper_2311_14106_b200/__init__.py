"""dmrgk — B200-native (sm_100a, FP64) H_eff·ψ and Davidson step of ab initio DMRG (arXiv 2311.14106).

The product is the C-ABI library ``_build/libdmrgk.so`` (sources in ``csrc/``, ABI in
``include/dmrgk.h``); ``dmrgk`` is its ctypes binding, ``problem`` sets problems up on the device,
``build`` compiles the library in-tree.  Importing this package does not need a GPU; every compute
call does, and fails loudly without one (there is no CPU or PyTorch fallback).
"""
from . import build as build_mod  # noqa: F401
from . import dmrgk  # noqa: F401

__all__ = ["dmrgk", "build_mod"]
