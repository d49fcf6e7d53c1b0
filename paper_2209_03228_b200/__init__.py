"""paper_2209_03228_b200 -- B200-native batched Landau Jacobian construction (arxiv 2209.03228 hot path).

`binding` is the ctypes layer over include/landau.h (liblandau_b200.so, hand-written CUDA for sm_100a);
`workloads` holds the seeded synthetic inputs; `build` compiles the library in-tree.  No CPU fallback exists:
`binding.load()` raises if the CUDA library is missing.
"""
