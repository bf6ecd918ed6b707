"""B200-native TPC track-model decoding (arXiv:2411.02206 §4): thin ctypes binding of libtmd.so (include/tmd.h).

There is no CPU fallback: importing `paper_2411_02206_b200.tmd` raises if the CUDA library cannot be built or loaded.
"""
