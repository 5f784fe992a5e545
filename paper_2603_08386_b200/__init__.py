"""DDHF hot path for B200 (sm_100a): CUDA kernels behind a C ABI (include/ddhf.h).

``workloads`` (input generators) imports nothing native; ``binding`` loads
``libddhf.so`` and raises if it is missing -- there is no CPU fallback.
"""
