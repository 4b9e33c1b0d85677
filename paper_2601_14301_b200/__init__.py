"""B200-native TRIMEG marker-push hot path (arxiv/paper_2601_14301).

`inputs`   seeded synthetic workloads (numpy only; shared with the test oracle)
`binding`  thin ctypes binding of the C-ABI library libtrimeg.so (CUDA, sm_100a)
`build`    compiles csrc/ into libtrimeg.so with nvcc

Importing the package does not load the CUDA library; `binding` does, and fails
loudly if it is missing -- there is no CPU fallback.
"""
__all__ = ["inputs", "binding", "build"]
