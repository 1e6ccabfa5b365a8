"""B200-native per-particle GRPIC hot path (arxiv/paper_2511_17701): CUDA kernels behind a C ABI.

    csrc/        the kernels and the extern "C" library (include/grpic.h)
    build.py     nvcc build step (sm_100a)
    grpic.py     thin ctypes binding with the ABI's names
    workloads.py seeded synthetic inputs shared by the CUDA path's callers and the oracle's callers
"""
