"""paper_1709_00821_b200 — librketd: the 1-D RKETD-FDTD leapfrog hot path of arxiv 1709.00821,
B200-native (hand-written sm_100a CUDA kernels behind a C ABI, include/rketd.h).

    from paper_1709_00821_b200 import rketd      # thin ctypes binding, same names as the C ABI
    from paper_1709_00821_b200 import workloads  # seeded synthetic inputs (no arithmetic of the method)

There is no CPU fallback: importing ``rketd`` loads ``librketd.so`` (built in-tree by
``python -m paper_1709_00821_b200.build``) and every compute call needs a CUDA device.
"""
__all__ = ["rketd", "workloads", "build"]
