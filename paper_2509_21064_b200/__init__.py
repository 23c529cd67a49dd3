"""B200-native (sm_100a) GDA hot path of PDBO (arxiv 2509.21064).

`workloads` (pure NumPy input generators) imports without the CUDA library; the binding in
`api` loads `lib/libgda_b200.so` lazily and fails loudly when it is missing.
"""
__all__ = ["workloads", "api"]
