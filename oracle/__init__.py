"""ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes access to oracle/stag_oracle.cpp (plain single-threaded C++, fp64).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package; the product (paper_1010_5433_b200/) never does and shares no code with it.
"""
from .api import (  # noqa: F401
    build, lib, set_threads, dslash, dslash_eo, dslash_oe, apply_A, mshift_cg, norm2,
    partial_fraction, dense_A, dense_solve, split_double, cg_polish, fermion_force,
)
