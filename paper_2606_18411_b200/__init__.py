"""paper_2606_18411_b200 -- B200-native (sm_100a) MRCQR: FP64 thin QR of tall-skinny matrices.

The product is the C-ABI library built from csrc/ (declared in include/mrcqr.h); `binding`
is a thin ctypes marshalling layer with the same names.  `inputs` holds the seeded synthetic
input generators used by tests, smoke() and bench.py.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs"]
