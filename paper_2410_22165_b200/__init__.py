"""B200-native batched EconoJax environment step (arXiv 2410.22165).

The product is the C-ABI library built from ``csrc/`` (declared in
``include/econojax.h``); ``binding`` is a thin ctypes marshalling layer with the
same names.  ``inputs`` holds the seeded synthetic workloads.  Nothing here falls
back to a CPU path: if the CUDA library is missing, ``binding.lib()`` raises.
"""

__all__ = ["binding", "inputs"]
