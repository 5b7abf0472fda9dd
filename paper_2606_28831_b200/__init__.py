"""hardkv-b200: B200-native (sm_100a) HARD-KV decode-step hot path (arxiv/paper_2606_28831).

`paper_2606_28831_b200.hardkv` is the thin ctypes binding over libhardkv.so (C ABI in
include/hardkv.h); importing it fails loudly if the CUDA library has not been built.
The seeded synthetic workloads live outside the package, in `workloads.synth` (numpy only).
"""
