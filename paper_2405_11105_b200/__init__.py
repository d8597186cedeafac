"""B200-native localized spatiotemporal EVD clutter filter (arXiv 2405.11105 hot path).

`synth` (numpy input generator) imports without the CUDA library; `lcf` (the ctypes binding of
liblcf.so) raises at first use if the library has not been built -- there is no CPU fallback.
"""
