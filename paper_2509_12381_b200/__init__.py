"""paper_2509_12381_b200 -- B200-native atom-ion trajectory integrator (aig).

``inputs``  : seeded synthetic workloads (NumPy only; shared with the test oracle).
``binding`` : thin ctypes binding of the C-ABI library ``libaig.so`` (include/aig.h).

The binding is imported lazily so that ``inputs`` stays usable on machines where the CUDA
library has not been built; every compute entry point fails loudly when it is missing.
"""
__all__ = ["inputs", "binding"]
__version__ = "0.1.0"
