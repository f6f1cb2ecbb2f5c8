"""B200-native (sm_100a) non-hydrostatic shallow-flow time step (arXiv 1706.04551).

`paper_1706_04551_b200.nh`      thin ctypes binding of the C-ABI library libnh_b200.so
                                (include/nh_b200.h); every step of the path runs in CUDA kernels.
`paper_1706_04551_b200.inputs`  seeded synthetic input generators (no method arithmetic).
`paper_1706_04551_b200.build`   nvcc build of csrc/ -> libnh_b200.so (in-tree).

Importing the package does not load the CUDA library; `nh` does, and fails loudly without it.
"""
__all__ = ["inputs", "nh", "build"]
