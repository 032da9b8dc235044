"""peek-b200: B200-native batched longest-prefix-match + pending-tree signals (PEEK, arxiv/paper_2607_02525).

The product is ``libpeek.so`` (hand-written sm_100a CUDA behind the C ABI of
``include/peek.h``); ``binding`` is the thin ctypes layer with the same names.  There is no CPU
fallback: ``binding`` raises if the CUDA library is missing.  (The synthetic workload generators
and the measurement probe live in the top-level ``harness`` package, not here.)
"""
__version__ = "0.1.0"
