"""fts-b200: B200-native hot path of polymer field-theoretic simulation (Delaney & Fredrickson, arXiv 1204.5434).

The product is the C-ABI library built from csrc/ (include/fts.h); `binding` is its thin Python
wrapper (argument marshalling only).  `inputs` holds the seeded synthetic workloads.
"""
