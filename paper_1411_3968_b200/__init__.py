"""B200-native tower trigger: time sort + L1/L2 trigger + event-window merge (arxiv 1411.3968 hot path).

`binding` holds the ctypes layer over libtt.so (include/tt.h); `workload` the seeded synthetic inputs.
Importing this package does not load CUDA; compute calls raise if libtt.so or a GPU is missing.
"""
