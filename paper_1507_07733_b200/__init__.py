"""paper_1507_07733_b200 -- B200-native per-station E-field unfolding (arXiv 1507.07733 hot path).

The product is the CUDA library libaera_unfold.so (csrc/, C ABI in include/aera_unfold.h).
`binding` is the thin ctypes layer with the same entry-point names; importing it loads the
library and fails loudly if it cannot be built or loaded. There is no CPU fallback.
"""
__all__ = ["binding", "build", "sharding"]
