"""B200-native density-fitted Coulomb/exchange (JK) build (arxiv 2505.03755, Eq. 14-17).

Thin Python binding over the C ABI in include/dfjk.h: argument marshalling only, every step of the
path runs in the CUDA kernels of csrc/.  PyTorch is used for device memory and streams.
"""
from .api import DFJK, DFJKError, get_jk, lib_path, load_library, selftest_dmma, small_jk_static

__all__ = ["DFJK", "DFJKError", "get_jk", "lib_path", "load_library", "selftest_dmma", "small_jk_static"]
