"""B200-native Vlasov full-step hot path of arXiv 1406.5445 (C-ABI library + thin binding).

`inputs` (seeded synthetic workloads) imports on any machine; `binding` loads the CUDA library
and fails loudly if it is missing -- there is no CPU fallback.
"""
__all__ = ["inputs", "binding"]
