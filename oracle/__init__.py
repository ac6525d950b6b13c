"""CPU oracle for the Barnes-Hut hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

`oracle/bh_oracle.c` is the plain single-threaded fp64 implementation written from the paper;
this package is its ctypes wrapper.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / `--impl reference` leg may import it.  It imports nothing from the CUDA package.
"""
from .bh_oracle import (OracleTree, keys, sort_perm, direct, direct_acc, build_library, MAC_BH86, MAC_BARNES94,  # noqa: F401
                        ewald_psi, ewald_corr, EwaldTable)
