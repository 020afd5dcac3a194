"""B200-native Cross-DEIM low-rank Poisson hot path (arxiv/paper_2607_06021).

`paper_2607_06021_b200.lrp`       -- thin ctypes binding of the C-ABI library (include/lrp.h)
`paper_2607_06021_b200.workloads` -- seeded synthetic inputs (shared with the oracle's tests)
`paper_2607_06021_b200.build`     -- nvcc build of csrc/ into liblrp.so (sm_100a)

Importing the package loads nothing; the CUDA library is loaded on first use of `lrp` and
raises if it is missing -- there is no CPU fallback.
"""
