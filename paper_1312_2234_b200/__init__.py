"""B200-native LBM + immersed-boundary hot path of arXiv:1312.2234 (Wu, Xu, Kim, Alber).

The package holds only what the path needs:

* ``csrc/``      -- hand-written CUDA kernels for sm_100a and the C-ABI (``include/plb.h``)
* ``binding``    -- thin ctypes binding with the same names as the C-ABI (argument marshalling only)
* ``workloads``  -- seeded synthetic input generators (no method arithmetic; shared with the oracle tests)
* ``build``      -- in-tree nvcc build of ``libplb.so``

Importing the package does not load the CUDA library; ``binding`` loads it on first use and
raises if it is missing (there is no CPU fallback).
"""

__all__ = ["binding", "workloads", "build"]
