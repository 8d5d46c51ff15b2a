"""B200-native (sm_100a, fp64) ADI sweep of the thin-film solver of arXiv:1806.10550.

`inputs` (seeded synthetic inputs) imports without the CUDA library; `tf` (the binding of the
C-ABI in include/tf.h) raises at first use if libtf_b200.so is missing -- there is no fallback.
"""
__all__ = ["inputs", "tf"]
