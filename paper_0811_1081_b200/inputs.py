"""Seeded synthetic inputs for the five BASELINE.json configs (and scaled-down siblings).

This module holds NONE of the method's arithmetic (no centring, no power iteration, no
Gram-Schmidt of the method, no deflation): it only draws the data matrices.  It is the one
module both the CPU oracle's tests and the CUDA path's tests / bench.py use, so both sides
consume the identical float32 array.  It imports neither `oracle` nor the CUDA binding.

Recipes (readings C14/C15 of SURVEY.md section 8(c)):
  * "N(0, 1e-3)" / "N(0, 1e-2)" in BASELINE.json is read as STANDARD DEVIATION.
  * the power-law spectrum is 1-based: s_k = 100/(k+1), k = 0..N-1; the others are 0-based.
  * U is made orthonormal AND zero-column-mean (draw G, remove its column means, then QR), so
    that column-mean centring is an exact-arithmetic no-op on the noise-free part and the
    prescribed spectrum survives centring.
  * QR sign convention: columns are flipped so that diag(R) > 0 (makes Q unique).
The paper's own workload (unseeded uniform [0,1) matrices, N = M/2, K = 10)
is available as kind="uniform" for the Fig.-1-shaped sweep.

All matrices are returned column-major (Fortran order, shape (M, N)), float32, NOT yet centred:
centring is the method's step S0 and is done by pca_center (CUDA) / oracle.center (oracle).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 8111081

ALGO_NIPALS = 0
ALGO_GS = 1


@dataclass(frozen=True)
class Config:
    name: str
    M: int
    N: int
    K: int
    eps: float
    max_iter: int
    algos: tuple          # subset of (ALGO_NIPALS, ALGO_GS)
    kind: str             # "spectrum" | "lowrank" | "scaled_gauss" | "uniform"
    spectrum: str = ""    # "geom" | "power" | "exp"  (kind == "spectrum")
    noise: float = 0.0    # standard deviation of the additive N(0, noise^2) term
    rank: int = 0         # kind == "lowrank": inner dimension of A B
    seed: int = BASE_SEED
    note: str = ""


# BASELINE.json `configs`, in order (cfg index 0..4 == "config 1..5" of SURVEY.md section 8).
CONFIGS = (
    Config("cfg1_256x64", 256, 64, 8, 1e-7, 10000, (ALGO_GS, ALGO_NIPALS), "spectrum",
           spectrum="geom", noise=1e-3, seed=BASE_SEED + 0, note="s_k = 10*0.8^k"),
    Config("cfg2_4096x1024", 4096, 1024, 32, 1e-7, 10000, (ALGO_GS,), "spectrum",
           spectrum="power", noise=1e-2, seed=BASE_SEED + 1, note="s_k = 100/(k+1); R = 16 MiB"),
    Config("cfg3_16384x4096", 16384, 4096, 64, 1e-7, 10000, (ALGO_NIPALS, ALGO_GS), "lowrank",
           noise=1e-3, rank=16, seed=BASE_SEED + 2, note="X = A B, collinear columns"),
    Config("cfg4_65536x2048", 65536, 2048, 128, 1e-7, 10000, (ALGO_GS,), "spectrum",
           spectrum="exp", noise=1e-2, seed=BASE_SEED + 3, note="s_k = 50*exp(-k/40); R = 512 MiB"),
    Config("cfg5_8192x512", 8192, 512, 512, 1e-8, 10000, (ALGO_GS,), "scaled_gauss",
           seed=BASE_SEED + 4, note="c_n = 1 + 9 u_n, K = N full decomposition"),
)


def scaled(cfg: Config, M: int, N: int, K: int | None = None, **kw) -> Config:
    """A smaller (or otherwise modified) sibling of a config: same recipe, same seed."""
    d = dict(cfg.__dict__)
    d.update(M=int(M), N=int(N), K=int(K if K is not None else min(cfg.K, N)),
             name=f"{cfg.name}_as_{M}x{N}")
    if d["kind"] == "lowrank":
        d["rank"] = min(cfg.rank, N)
    d.update(kw)
    return Config(**d)


def spectrum_values(kind: str, n: int) -> np.ndarray:
    k = np.arange(n, dtype=np.float64)
    if kind == "geom":
        return 10.0 * 0.8 ** k
    if kind == "power":
        return 100.0 / (k + 1.0)
    if kind == "exp":
        return 50.0 * np.exp(-k / 40.0)
    raise ValueError(f"unknown spectrum {kind!r}")


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(int(seed)))


def random_orthonormal(rng: np.random.Generator, rows: int, cols: int, zero_mean: bool) -> np.ndarray:
    """rows x cols matrix with orthonormal columns from QR of N(0,1) draws (float64).

    zero_mean=True removes the column means of the draws first, so every column of Q sums to
    zero (Q's columns span the column space of the de-meaned draws)."""
    G = rng.standard_normal((rows, cols))
    if zero_mean:
        G -= G.mean(axis=0, keepdims=True)
    Q, Rf = np.linalg.qr(G, mode="reduced")
    sgn = np.sign(np.diag(Rf))
    sgn[sgn == 0] = 1.0
    Q *= sgn[None, :]
    return Q


@dataclass
class Problem:
    cfg: Config
    X: np.ndarray                                  # (M, N) float32, Fortran order, not centred
    truth: dict = field(default_factory=dict)      # what the recipe prescribes (s, U, V) if any


def generate(cfg: Config, keep_factors: bool = False) -> Problem:
    """Draw the data matrix of a config.  Deterministic in cfg (seed, sizes, recipe)."""
    M, N = cfg.M, cfg.N
    rng = _rng(cfg.seed)
    truth: dict = {}
    if cfg.kind == "spectrum":
        if M < N:
            raise ValueError("spectrum recipe needs M >= N")
        U = random_orthonormal(rng, M, N, zero_mean=True)
        V = random_orthonormal(rng, N, N, zero_mean=False)
        s = spectrum_values(cfg.spectrum, N)
        X = (U * s[None, :]) @ V.T
        truth["s"] = s
        if keep_factors:
            truth["U"], truth["V"] = U, V
        del U
    elif cfg.kind == "lowrank":
        A = rng.standard_normal((M, cfg.rank))
        B = rng.standard_normal((cfg.rank, N))
        X = A @ B
    elif cfg.kind == "scaled_gauss":
        X = rng.standard_normal((M, N))
        u = rng.random(N)
        X *= (1.0 + 9.0 * u)[None, :]
        truth["col_scale"] = 1.0 + 9.0 * u
    elif cfg.kind == "uniform":
        X = rng.random((M, N))                    # paper's workload
    else:
        raise ValueError(f"unknown kind {cfg.kind!r}")
    if cfg.noise > 0.0:
        rows = max(1, (1 << 24) // max(N, 1))     # add the noise in slabs to bound memory
        for m0 in range(0, M, rows):
            m1 = min(M, m0 + rows)
            X[m0:m1] += cfg.noise * rng.standard_normal((m1 - m0, N))
    Xf = np.asfortranarray(X.astype(np.float32))
    return Problem(cfg=cfg, X=Xf, truth=truth)


def config(i: int) -> Config:
    """BASELINE.json configs[i], i = 0..4."""
    return CONFIGS[i]
