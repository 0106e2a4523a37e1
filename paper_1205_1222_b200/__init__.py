"""B200-native Ahmad-Cohen regular force (arXiv 1205.1222): Hermite j-predictor, regular force + jerk,
neighbour lists.  The compute path is the C-ABI CUDA library in csrc/ (include/nbreg.h); this package is
a thin ctypes binding plus the seeded input generators."""
