"""B200-native floating-mean Lomb-Scargle hot path (arXiv:2409.08090) — C-ABI library + thin binding.

`binding` mirrors include/ls.h (ls_plan / ls_execute / ls_destroy ...); `workloads` holds the seeded
synthetic inputs (numpy only, none of the method's arithmetic); `build` compiles the library in-tree.
"""
