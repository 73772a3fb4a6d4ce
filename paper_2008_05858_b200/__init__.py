"""B200-native echellogram rendering: the hot path of the end-to-end spectrograph simulator of arXiv 2008.05858.

``binding``   ctypes binding of the C-ABI library ``libe2e.so`` (``include/e2e.h``)
``workloads`` seeded synthetic inputs (shared with the CPU oracle; holds none of the method's arithmetic)
``build``     in-tree nvcc build of ``libe2e.so`` for sm_100a
"""
__all__ = ["binding", "workloads", "build"]
