"""B200-native RAPTOR hot path (arXiv:1801.10452): per-pixel Kerr null geodesics fused with
covariant radiative transfer, as hand-written FP64 CUDA for sm_100a behind a C ABI.

``scenes``  -- seeded synthetic inputs (data only; also handed to the test oracle)
``binding`` -- thin ctypes binding of include/raptor.h (argument marshalling only)
"""
__all__ = ["scenes", "binding"]
