"""B200-native bead-rod Brownian dynamics with hydrodynamic interactions (arXiv 2208.06559 hot path).

The product is ``libbd.so`` (hand-written sm_100a CUDA behind the C ABI of ``include/bd.h``);
``paper_2208_06559_b200.binding`` is argument marshalling only.  Nothing here imports ``oracle``.
"""
__all__ = ["workloads"]
