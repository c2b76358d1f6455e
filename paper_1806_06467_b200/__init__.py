"""fresnel-b200: B200-native plane-to-plane Fresnel propagation (the hot path of arXiv 1806.06467).

``inputs``  -- seeded synthetic workload generators (pure numpy, no method arithmetic).
``binding`` -- thin ctypes face of ``libfresnel.so`` (the C ABI in include/fresnel.h).
"""
__all__ = ["inputs", "binding"]
