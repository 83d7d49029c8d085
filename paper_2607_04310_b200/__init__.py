"""B200-native PSDF hot path (arxiv/paper_2607_04310): C-ABI library + thin binding.

`paper_2607_04310_b200.psdf` is the binding over `libpsdf.so` (CUDA, sm_100a);
`paper_2607_04310_b200.workloads` holds the seeded input recipes only.
"""
