"""B200-native Kohn-Sham H|psi> and Taylor-4 real-time TDDFT step (arXiv:2106.03872 hot path).

The package holds three things only:

* ``workloads``  -- seeded synthetic input generators (no method arithmetic; shared with the tests' oracle),
* ``binding``    -- thin ctypes binding of the C-ABI library ``libtdh.so`` (``include/tdh.h``),
* ``csrc/``      -- the CUDA sources of that library (built in-tree by ``build.py``).

Importing the package does not load the CUDA library; ``binding`` does, and fails loudly
if it is missing.  There is no CPU fallback.
"""

__all__ = ["workloads", "binding", "build"]
