"""B200-native (sm_100a) Monte Carlo 2->2 collision term of the relativistic Boltzmann equation (arXiv:1912.04457).

The product is the C-ABI shared library paper_1912_04457_b200/libbz.so (include/bz.h); this package is its thin
Python binding (argument marshalling only).  PyTorch provides device memory and streams, nothing else.
"""
from .bz import Boltzmann, lib, LIB_PATH  # noqa: F401
