"""B200-native assembly of the implicit two-fluid finite-volume residual and its BSR Jacobian.

``workloads``  seeded synthetic meshes and states (shared with the test oracle; no method arithmetic)
``api``        thin binding of the C ABI in include/tfa.h (needs torch + the built libtfa.so)
``build``      nvcc build of csrc/ -> libtfa.so
"""
__all__ = ["workloads", "api", "build"]
