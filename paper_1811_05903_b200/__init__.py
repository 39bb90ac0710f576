"""steps-b200: B200-native StePS hot path (direct-summation forces + comoving KDK).

The product is the C-ABI library built from csrc/ (include/steps.h); `steps` is the thin
ctypes binding with the same names.  Nothing here imports oracle/ (test infrastructure)."""
__version__ = "0.1.0"
