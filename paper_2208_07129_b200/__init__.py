"""B200-native (sm_100a) matrix-free FE Helmholtz multivector apply + Chebyshev filter.

Hot path of arXiv 2208.07129 behind a C-ABI (`include/fe_mf.h`); this package is only the
ctypes binding (`binding.py`) and the seeded input generators (`inputs.py`).  Importing the
package does not load the CUDA library; `binding.lib()` does and fails loudly if it is missing.
"""
__all__ = ["binding", "inputs"]
