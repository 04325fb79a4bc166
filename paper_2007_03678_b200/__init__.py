"""B200-native (sm_100a) hot path of AutoDock-GPU-style LGA docking (arxiv 2007.03678).

`workloads` holds the seeded synthetic input generators; `binding` is the thin ctypes layer over the
C-ABI library (include/adock.h) whose CUDA kernels do every step of the path.
"""
