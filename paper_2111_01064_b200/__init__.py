"""B200-native batched LISA MBHB log-likelihood (arXiv:2111.01064 hot path).

`paper_2111_01064_b200.binding`  — thin ctypes binding over the C-ABI library (include/ll.h)
`paper_2111_01064_b200.workloads` — seeded synthetic inputs shared by the oracle and the CUDA path
`paper_2111_01064_b200.build`     — nvcc build of csrc/ into libll_b200.so (sm_100a)
"""
__all__ = ["binding", "workloads", "build"]
