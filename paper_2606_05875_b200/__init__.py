"""B200-native (sm_100a) implementation of the QCFuse per-layer selective-recompute step (arxiv 2606.05875).

`binding` is the ctypes face of the C-ABI library libqcf.so (include/qcf.h); `build` compiles it in-tree;
`inputs` synthesises seeded workloads; `device` puts them into device buffers for tests and bench.py.
"""
