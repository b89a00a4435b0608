"""paper_2303_08123_b200 -- B200-native batched fitness evaluation for the GPU-GA
radiotherapy-protocol search of arxiv 2303.08123 (hot path only).

Importing the package is cheap and loads no native code; `binding.load()` loads
the in-tree CUDA library and raises if it is missing (there is no CPU fallback).
"""
