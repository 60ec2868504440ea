"""CPU oracle for arxiv 0811.1081 (NIPALS-PCA / GS-PCA) -- test infrastructure only.

See oracle/pca_oracle.cpp for the algorithm (cited line by line against PAPER.md) and
oracle/pca_oracle.py for the ctypes binding.  Nothing under paper_0811_1081_b200/ imports this.
"""
from .pca_oracle import (ALGO_GS, ALGO_NIPALS, OracleResult, build, center, center_eq1,
                         jacobi_eigh, num_threads, pca, set_num_threads)

__all__ = ["ALGO_GS", "ALGO_NIPALS", "OracleResult", "build", "center", "center_eq1",
           "jacobi_eigh", "num_threads", "pca", "set_num_threads"]
