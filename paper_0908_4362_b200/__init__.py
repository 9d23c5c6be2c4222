"""paper_0908_4362_b200 -- B200-native relaxing-TVD ideal-MHD update (hot path of arxiv/paper_0908_4362).

``paper_0908_4362_b200.inputs``  seeded synthetic initial states (no method arithmetic).
``paper_0908_4362_b200.binding`` thin ctypes binding of the C ABI in include/mhd.h (libmhd.so); importing
it fails loudly when the CUDA library has not been built -- there is no CPU fallback.
"""
__all__ = ["inputs", "binding"]
