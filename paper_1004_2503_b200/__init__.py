"""B200-native ATON hot path (explicit M1 radiative transfer + H chemistry) behind a C ABI.

`workloads` (seeded synthetic inputs) imports without the CUDA library; everything in `aton`
needs `libaton.so` (built by `paper_1004_2503_b200.build`) and fails loudly without it.
"""
__all__ = ["aton", "workloads", "build"]
