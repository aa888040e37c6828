"""Looking Forward (arxiv 2402.14670) track following, B200-native hot path.

Public API: :class:`paper_2402_14670_b200.binding.LookingForward` (thin ctypes binding over the
C-ABI library declared in ``include/lf.h``).  ``datagen`` holds the seeded input generators.
The CUDA library is loaded lazily and loudly: there is no CPU fallback.
"""
__all__ = ["datagen"]
