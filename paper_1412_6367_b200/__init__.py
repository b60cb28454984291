"""B200-native 1D azimuthal integration (hot path of arxiv 1412.6367): C-ABI CUDA library + thin Python binding.

`paper_1412_6367_b200.binding` marshals arguments to `libazint.so` (include/azint.h); every step of the path runs in
the CUDA kernels under `csrc/`.  `paper_1412_6367_b200.workloads` holds the seeded synthetic inputs.  There is no CPU
fallback: using the binding without the compiled library, or without a CUDA device, raises.
"""
__all__ = ["binding", "workloads", "build"]
