"""B200-native worldline numerics (Loop Cloud Method) hot path, arXiv:1407.7486.

`paper_1407_7486_b200.api` is the thin binding of the C-ABI library built from
`csrc/` (include/wl.h); importing it fails loudly if the CUDA library has not
been built.  `paper_1407_7486_b200.inputs` holds the seeded workload shapes.
"""
