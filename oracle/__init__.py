"""CPU oracle for the DF-JK path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It wraps oracle/dfjk_oracle.c (plain C loops, fp64, Eq. 12-17) and
oracle/ao2mo_oracle.c (Eq. 18-21) with ctypes
and numpy; it shares nothing with paper_2505_03755_b200 and never imports it.
"""
from .api import (ao2mo, ao2mo_bruteforce, ao2mo_sample, bruteforce, density, get_jk, get_jk_inputs, get_k_dform, num_threads, sample,
                  unpack_slice)

__all__ = ["ao2mo", "ao2mo_bruteforce", "ao2mo_sample", "bruteforce", "density", "get_jk", "get_jk_inputs", "get_k_dform", "num_threads",
           "sample", "unpack_slice"]
