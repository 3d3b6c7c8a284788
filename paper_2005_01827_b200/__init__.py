"""mbhl: B200-native batched LISA MBHB log-likelihood (hot path of arXiv:2005.01827).

The product is the C-ABI library built from csrc/ (include/mbhl.h); `binding`
marshals arguments to it with ctypes and has no fallback.  `workloads` holds the
seeded synthetic input generators (no method arithmetic).
"""
