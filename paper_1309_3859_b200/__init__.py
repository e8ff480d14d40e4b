"""B200-native hot path of arXiv:1309.3859 (compact U(1) multilevel Monte Carlo).

The product is the C-ABI library ``libul.so`` (see ``include/ul.h``) built from the CUDA
sources in ``csrc/``; ``ul`` is its thin ctypes binding (argument marshalling only).
"""
from . import ul  # noqa: F401
from .ul import Lattice, UlError  # noqa: F401
