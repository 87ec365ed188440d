"""B200-native parallel-tempering sweep of the 1-D long-range q-state Potts model
(arXiv 1308.5426).  `paper_1308_5426_b200.pt` is the thin binding over the C-ABI
library `libpt.so` (include/pt.h); `paper_1308_5426_b200.inputs` holds the seeded
workload recipes.  Nothing here falls back to a CPU path: importing `.pt` without a
built `libpt.so` raises."""
__all__ = ["inputs", "pt", "pt_math", "build", "shard"]
