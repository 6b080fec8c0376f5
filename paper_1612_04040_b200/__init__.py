"""B200-native narrow-band level-set hot path (arxiv/paper_1612_04040).

The product is the C-ABI library `libls.so` (include/ls.h, csrc/*.cu); this package is the thin
Python binding (argument marshalling only) plus the seeded input generators.
"""
