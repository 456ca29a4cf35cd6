"""paper_2502_07060_b200 -- B200-native Berends-Giele recursion (arXiv:2502.07060).

    binding   ctypes binding of libbg_b200.so (CUDA kernels, include/bg.h)
    inputs    seeded synthetic kinematics (shared with the test oracle; no BG arithmetic)
    build     in-tree nvcc build of the library

Importing the package does not load the CUDA library; `binding.load()` does, and raises
if it is missing (there is no CPU fallback).
"""
__all__ = ["binding", "inputs", "build"]
