"""B200-native MAC projection of MAESTROeX (arXiv:1910.12979): thin Python binding over the C-ABI
library `libmaestro_mac.so` (hand-written sm_100a CUDA kernels, include/maestro_mac.h).

    from paper_1910_12979_b200 import mac        # ctypes binding (loads the CUDA library)
    from paper_1910_12979_b200 import workloads  # seeded synthetic inputs (numpy only)

Nothing here falls back to a CPU implementation: `mac` raises if the CUDA library is missing.
"""
__all__ = ["mac", "workloads"]
