"""B200-native RA-MPPI hot path (arXiv 2209.12842): C-ABI CUDA library + thin Python binding.

    from paper_2209_12842_b200 import workloads, binding
    from paper_2209_12842_b200.controller import RaMppi      # needs torch + a B200

Importing the package does not load the CUDA library; the first binding call does, and it
raises if libra_mppi.so has not been built.  There is no CPU fallback.
"""
__all__ = ["workloads", "binding", "build"]
