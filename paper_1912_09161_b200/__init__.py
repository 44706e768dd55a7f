"""B200-native VELO pixel reconstruction hot path of Allen's HLT1 (arXiv:1912.09161).

`binding` — ctypes layer over the C ABI of include/allen_velo.h (CUDA kernels in csrc/, sm_100a only, no fallback).
`workload` — seeded synthetic inputs (geometry G0, event generator, raw packer).
`build`    — builds the extension in-tree.
"""
__all__ = ["binding", "workload", "build"]
