"""B200-native hot path of Cleanba's actor-learner method (arXiv 2310.00036).

`synth` holds the seeded input generators (no method arithmetic); `binding` is the thin ctypes
layer over the C-ABI CUDA library in csrc/ (include/cleanba.h).  Nothing here falls back to CPU.
"""
