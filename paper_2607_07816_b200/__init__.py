"""B200-native sparse, truncated state-vector gate engine (arxiv/paper_2607_07816).

  paper_2607_07816_b200.engine     thin ctypes binding of the C-ABI library
                                   (include/sparse_sv.h); fails loudly if the CUDA
                                   library has not been built
  paper_2607_07816_b200.workloads  seeded synthetic circuit generators (inputs only)
  paper_2607_07816_b200.qasm       OpenQASM 2.0 reader -> the same gate records (inputs only)
  paper_2607_07816_b200.build      nvcc build of csrc/ -> libsparse_sv.so (sm_100a)
"""
__all__ = ["engine", "workloads", "qasm", "build"]
