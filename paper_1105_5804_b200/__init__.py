"""paper_1105_5804_b200 -- Swendsen-Wang / Wolff cluster updates of the 2D Ising / Potts model, B200-native.

The product is the C-ABI library ``libswb200.so`` (include/swb200.h, csrc/*.cu, sm_100a); this package is its thin
Python binding (argument marshalling only).  Nothing is loaded at import time; ``binding.lib()`` loads the
shared library on first use and raises if it is missing -- there is no CPU fallback.
"""
__all__ = ["binding", "inputs", "build"]
