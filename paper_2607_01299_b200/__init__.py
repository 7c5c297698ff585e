"""B200-native HYPIC linear-attention hot path: segment encode -> (E, T), composition S <- S.T_i + E_i.

The product is the C-ABI library ``libhypic.so`` (``include/hypic.h``, ``csrc/``); ``binding`` is the thin
argument-marshalling layer with the same entry-point names, ``workloads`` the seeded synthetic inputs.
Nothing here falls back to the CPU: calling an op without the built CUDA library raises.
"""
__version__ = "0.1.0"
