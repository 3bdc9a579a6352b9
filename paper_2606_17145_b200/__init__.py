"""paper_2606_17145_b200 -- B200-native TreePM short-range gravity (tree build + walk).

`workloads` (seeded inputs) imports without the CUDA library; everything in `binding`
needs `libogtree.so` and fails loudly when it is missing (there is no CPU fallback).
"""
