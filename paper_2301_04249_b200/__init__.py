"""B200-native RT-EOM-CCSD hot path (arXiv:2301.04249): C-ABI library ``librtcc.so`` + thin binding.

``inputs`` (seeded synthetic workloads) imports nothing heavy; ``rtcc`` (the binding) loads the CUDA
library on first use and raises loudly if it is missing -- there is no CPU fallback.
"""
__all__ = ["inputs", "rtcc"]
