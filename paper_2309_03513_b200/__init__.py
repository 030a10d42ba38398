"""B200-native TDA Liouville operator of plane-wave hybrid LR-TDDFT (arXiv 2309.03513).

`paper_2309_03513_b200.binding` is the ctypes face of the C ABI in include/tddft.h (CUDA only, no CPU
fallback); `paper_2309_03513_b200.build` compiles the library in-tree.  The seeded synthetic input generators shared
by the tests, the oracle and bench.py live outside the package (synthetic_inputs.py).
"""
