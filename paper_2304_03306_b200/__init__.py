"""B200-native (sm_100a) pseudospectral TTSH step of arXiv:2304.03306 behind a C ABI.

``paper_2304_03306_b200.ttsh``      thin ctypes binding of include/ttsh.h (loads csrc/libttsh.so)
``paper_2304_03306_b200.workloads`` seeded synthetic inputs (shared with the test oracle)
Nothing is imported eagerly: the binding fails loudly when the CUDA library is missing.
"""
__all__ = ["ttsh", "workloads"]
