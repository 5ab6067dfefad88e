"""B200-native w-projection convolutional gridder (hot path of arxiv 1905.03213).

``paper_1905_03213_b200.wpgrid`` is the thin ctypes binding over the C-ABI
library ``libwpgrid.so`` (include/wpgrid.h); ``paper_1905_03213_b200.synth``
holds the seeded input generators.  Nothing is imported eagerly so that
``synth`` can be used without the CUDA library.
"""
__all__ = ["wpgrid", "synth"]
