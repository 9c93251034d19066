"""smolgp-b200: B200-native integrated-GP inference (arXiv:2601.02527) behind a C ABI.

`workloads` (seeded synthetic inputs) imports without CUDA; the binding (`smolgp`) loads the
in-tree CUDA shared library lazily and fails loudly if it is missing.
"""
