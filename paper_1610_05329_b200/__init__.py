"""paper_1610_05329_b200 -- B200-native split-step Crank-Nicolson step of the 3-D dipolar
Gross-Pitaevskii equation (arXiv:1610.05329).

The product is the C-ABI library declared in include/dgpe.h (built from csrc/ into
libdgpe.so); `binding` is the thin ctypes layer over it, `inputs` the seeded input generators.
Nothing here falls back to a CPU implementation: without the built CUDA library every call raises.
"""
__all__ = ["binding", "inputs", "build"]
