"""mphv: B200-native (sm_100a) kinetic Vlasov sweeps and velocity moments.

``inputs`` -- seeded synthetic workloads (numpy only, shared with the test oracle).
``mphv``   -- thin ctypes binding of the C-ABI library built from ``csrc/`` (loaded
              lazily; it raises if the CUDA library is missing -- there is no CPU fallback).
"""
__all__ = ["inputs", "mphv"]
