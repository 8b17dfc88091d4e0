"""B200-native batched per-walker step of k-point ph-AFQMC (arxiv 2003.09468).

The compute path is the C-ABI CUDA library `libafqmc.so` (sources in `csrc/`, header
`include/afqmc.h`); `binding` is argument marshalling only.  Importing this package does not
load the library; `paper_2003_09468_b200.binding.lib()` does, and fails loudly if it is missing.
"""
__all__ = ["synth", "binding"]
