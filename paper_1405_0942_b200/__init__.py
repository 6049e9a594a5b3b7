"""B200-native Lagrangian magneto-frictional relaxation step (arxiv 1405.0942, the GLEMuR method).

Sub-modules
-----------
inputs : seeded, closed-form synthetic workloads (numpy only; none of the method's arithmetic).
mr     : thin ctypes binding over the C-ABI library ``libmr.so`` (include/mr.h). Importing it
         fails loudly when the CUDA library has not been built; there is no CPU fallback.
build  : nvcc build of ``csrc/`` into ``libmr.so`` (sm_100a).

Nothing is imported eagerly so that ``inputs`` stays usable by the CPU oracle tests.
"""

__all__ = ["inputs", "mr", "build"]
