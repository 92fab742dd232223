"""B200-native PRISM / multislice STEM simulation hot path (arXiv 1706.08563).

``paper_1706_08563_b200.prism``     thin ctypes binding of the C-ABI library
                                    (``include/prism.h``); every step runs in the
                                    CUDA kernels under ``csrc/``.  Importing it
                                    fails loudly if the library is not built.
``paper_1706_08563_b200.workloads`` seeded synthetic inputs (no method arithmetic).
``paper_1706_08563_b200.build``     nvcc build of ``libprism_b200.so`` (sm_100a).
"""
__all__ = ["workloads"]
