"""B200-native MeshBlockPack hydro stage (arXiv 2409.16053 hot path).

`ak` is the thin binding over the C-ABI library built from csrc/ (include/ak.h); `inputs` holds the
seeded synthetic workloads.  Nothing here falls back to a CPU implementation: using `ak` without the
compiled CUDA library raises.
"""
__all__ = ["ak", "inputs"]
