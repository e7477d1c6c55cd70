"""B200-native resampling F-statistic hot path (arXiv:2201.00451, steps iii-vii).

`synth` holds the seeded input generators; `binding` is the thin ctypes layer
over the C-ABI library built from `csrc/` (see include/fstat.h).
"""
