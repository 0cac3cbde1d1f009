"""B200-native CATAPULT hot path (arxiv/paper_2604_07617): tricubic field tables, fp64 DP5
guiding-centre tracer and Monte-Carlo estimate behind the C-ABI of include/catapult.h.

`workloads` (numpy-only seeded inputs) imports without the CUDA library; `binding` loads
libcatapult.so and fails loudly when it is missing.
"""
