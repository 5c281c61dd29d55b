"""libfasttg: B200-native temporal-attention message passing (FAST, arxiv/paper_2607_05095 §4.3).

The product is the C-ABI shared library ``libfasttg.so`` (hand-written sm_100a CUDA; see
``include/fasttg.h``).  ``binding`` is a thin ctypes marshalling layer with the same names.
Importing this package does not load the library; ``binding.lib()`` does and fails loudly if it
is missing.
"""
__all__ = ["binding", "build"]
