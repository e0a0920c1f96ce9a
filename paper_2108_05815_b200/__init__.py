"""necsim-b200: the Independent algorithm's hot path (arxiv 2108.05815) on one B200.

`paper_2108_05815_b200.necsim` is the ctypes binding of the C-ABI in include/necsim.h (loads
csrc/libnecsim_b200.so, needs a GPU). `paper_2108_05815_b200.inputs` holds the seeded synthetic input
generators shared by the tests, the oracle and bench.py; it contains none of the method's arithmetic.
Nothing is imported eagerly so that `inputs` can be used without the CUDA library.
"""
__all__ = ["inputs", "necsim"]
