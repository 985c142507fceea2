"""B200-native fictitious-wave-domain 3-D CSEM FDTD (hot path of libEMM, arxiv 2304.00233).

`paper_2304_00233_b200.emm` is the thin ctypes binding of the C-ABI library (include/emm.h);
`paper_2304_00233_b200.workloads` holds the seeded synthetic inputs.  Nothing here falls back
to a CPU implementation: the binding raises if libemm_b200.so is missing.
"""
__all__ = ["emm", "workloads"]
