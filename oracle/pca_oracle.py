"""ctypes binding of the CPU oracle (oracle/pca_oracle.cpp) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the CUDA package and the CUDA package never imports it.

All matrices are numpy float64, column-major (Fortran order), the paper's id(m,n,ld)=n*ld+m
(PAPER.md:399).  Inputs given as float32 are widened exactly to float64 first.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pca_oracle.cpp")
_LIB = os.path.join(_HERE, "libpca_oracle.so")

ALGO_NIPALS = 0
ALGO_GS = 1


def build(force: bool = False) -> str:
    """Compile oracle/pca_oracle.cpp -> oracle/libpca_oracle.so with g++ (no CUDA)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        # PCA_ORACLE_LIB: tests/test_oracle_mutants.py points this at a deliberately broken build of pca_oracle.cpp to
        # check that the pins notice (mutation test of the pins); never set otherwise.
        lib = ctypes.CDLL(os.environ.get("PCA_ORACLE_LIB") or build())
        i64, f64, i32 = ctypes.c_int64, ctypes.c_double, ctypes.c_int
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        lib.oracle_num_threads.restype = i32
        lib.oracle_set_num_threads.argtypes = [i32]
        lib.oracle_center.argtypes = [dp, i64, i64]
        lib.oracle_center_eq1.argtypes = [dp, i64, i64]
        lib.oracle_pca.argtypes = [dp, i64, i64, i32, f64, i32, i32, dp, dp, dp, ip, dp]
        lib.oracle_pca_ex.argtypes = [dp, i64, i64, i32, f64, i32, i32, i32, dp, dp, dp, ip, dp]
        lib.oracle_pca_ex2.argtypes = [dp, i64, i64, i32, f64, i32, i32, i32, i32, dp, dp, dp, ip, dp]
        lib.oracle_jacobi_eigh.argtypes = [dp, i32, dp, dp, i32, f64]
        _lib = lib
    return _lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _as_f64_colmajor(X) -> np.ndarray:
    X = np.asarray(X)
    if X.ndim != 2:
        raise ValueError("X must be 2-D (M x N)")
    return np.array(X, dtype=np.float64, order="F", copy=True)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def center(X) -> np.ndarray:
    """Column-mean centring (reading C1).  Returns a new float64 F-ordered array."""
    Xc = _as_f64_colmajor(X)
    M, N = Xc.shape
    if _load().oracle_center(_dptr(Xc), M, N) != 0:
        raise ValueError("oracle_center: invalid arguments")
    return Xc


def center_eq1(X) -> np.ndarray:
    """Literal eq. (1): subtract the mean column.  Non-default."""
    Xc = _as_f64_colmajor(X)
    M, N = Xc.shape
    if _load().oracle_center_eq1(_dptr(Xc), M, N) != 0:
        raise ValueError("oracle_center_eq1: invalid arguments")
    return Xc


@dataclass
class OracleResult:
    T: np.ndarray        # M x K scores, ||T[:,k]|| = lam[k]
    P: np.ndarray        # N x K unit loadings
    lam: np.ndarray      # K
    iters: np.ndarray    # K int32
    R: np.ndarray | None  # M x N residual (if requested)


def pca(X, K: int, eps: float = 1e-7, max_iter: int = 10000, algo: int = ALGO_GS,
        want_residual: bool = True, test_mode: int = 0, gs_passes: int = 1) -> OracleResult:
    """Run the oracle's NIPALS-PCA / GS-PCA on an (already centred) M x N matrix.
    test_mode 0: the listings' strict relative test; 1: the text's absolute test.
    gs_passes 1: one classical Gram-Schmidt projection per side per pass (the listings); 2: CGS2."""
    Xd = _as_f64_colmajor(X)
    M, N = Xd.shape
    T = np.zeros((M, K), dtype=np.float64, order="F")
    P = np.zeros((N, K), dtype=np.float64, order="F")
    lam = np.zeros(K, dtype=np.float64)
    iters = np.zeros(K, dtype=np.int32)
    R = np.zeros((M, N), dtype=np.float64, order="F") if want_residual else None
    rc = _load().oracle_pca_ex2(_dptr(Xd), M, N, int(K), float(eps), int(max_iter), int(algo), int(test_mode), int(gs_passes),
                               _dptr(T), _dptr(P), _dptr(lam),
                            iters.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                            _dptr(R) if R is not None else None)
    if rc != 0:
        raise ValueError("oracle_pca: invalid arguments")
    return OracleResult(T=T, P=P, lam=lam, iters=iters, R=R)


def jacobi_eigh(A, max_sweeps: int = 60, tol: float = 1e-15):
    """Cyclic Jacobi eigen-decomposition of a symmetric matrix.  Returns (w, Vec, sweeps)."""
    Ad = _as_f64_colmajor(A)
    n = Ad.shape[0]
    if Ad.shape[1] != n:
        raise ValueError("A must be square")
    w = np.zeros(n, dtype=np.float64)
    V = np.zeros((n, n), dtype=np.float64, order="F")
    sweeps = _load().oracle_jacobi_eigh(_dptr(Ad), n, _dptr(w), _dptr(V), int(max_sweeps), float(tol))
    if sweeps < 0:
        raise ValueError("oracle_jacobi_eigh: invalid arguments")
    return w, V, sweeps
