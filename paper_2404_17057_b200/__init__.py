"""B200-native compressible-flow MPM particle-grid cycle (arXiv 2404.17057).

`paper_2404_17057_b200.inputs`  seeded synthetic workloads (numpy only, no CUDA needed)
`paper_2404_17057_b200.binding` thin ctypes binding over the C-ABI library libmpm_b200.so (CUDA, sm_100a)

Importing the package does not load the CUDA library; `binding.load()` does and fails loudly if it is missing.
"""
__all__ = ["inputs", "binding"]
