"""okdirac: B200-native Oktay-Kronfeld Dirac apply + BiCGStab (arXiv:1311.5029, Eq. 2.2).

The package holds only what the hot path needs:

* ``csrc/``     hand-written sm_100a CUDA kernels and the C-ABI (``include/ok.h``)
* ``binding``   thin ctypes binding with the same names as the C-ABI (marshalling only)
* ``inputs``    seeded synthetic input generators (no arithmetic of the method)
* ``build``     in-tree nvcc build of ``libokdirac.so``

Importing the package never loads the CUDA library; ``binding.lib()`` does, and raises
``RuntimeError`` if ``libokdirac.so`` is missing.  There is no CPU fallback.
"""

__all__ = ["binding", "inputs", "build"]
