"""paper_2504_16446_b200 — B200-native (sm_100a) hot path of SAXS/WAXS tensor tomography (arxiv 2504.16446).

`mm`     thin ctypes binding of the C ABI in include/mm.h (libmm.so; no CPU fallback)
`synth`  seeded synthetic inputs shared by the tests, the bench and the oracle's callers
`build`  nvcc build of libmm.so (python -m paper_2504_16446_b200.build)
"""
