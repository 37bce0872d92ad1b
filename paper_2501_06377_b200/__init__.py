"""B200-native time-stepping hot path of the HipFT surface-flux-transport model (arxiv 2501.06377).

`paper_2501_06377_b200.hft`        ctypes binding of the C-ABI library (csrc/ -> libhft.so); importing it
                                   loads the CUDA library and fails loudly if it is missing.
`paper_2501_06377_b200.workloads`  seeded synthetic inputs shared by the CUDA path and the CPU oracle
                                   (no method arithmetic).
Nothing is imported eagerly so that `workloads` can be used without the CUDA library.
"""
__all__ = ["hft", "workloads", "build"]
