"""B200-native (sm_100a) contracted Clebsch-Gordan tensor products (SCALE-CG hot path).

The compute lives in csrc/ (hand-written CUDA behind the C ABI of include/cgtp.h); `binding`
marshals torch tensors into that ABI.  Importing this package does not load the CUDA library;
the first call into `binding` does, and fails loudly if it is missing.
"""
__version__ = "0.1.0"
