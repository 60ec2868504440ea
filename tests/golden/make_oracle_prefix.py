"""Write the stored full-size oracle results under tests/golden/ (calls ONLY oracle/ and the
seeded input generator; never the CUDA path).

    python tests/golden/make_oracle_prefix.py [cfg_index ...]        # default: all five configs

For each BASELINE.json config (paper_0811_1081_b200.inputs.CONFIGS) and each algorithm it lists,
the double-precision oracle (oracle/pca_oracle.cpp, the paper's algorithm step by step) is run
on the FULL-SIZE seeded input for the first K_s components.  Components are extracted one after
the other, so the first K_s components of a K-component solve are exactly the
K_s-component solve: the stored prefix is what the full run would return for those components.
K_s is the whole K for configs 1-4 (configs 3 and 4: one oracle pass streams 1-2 GiB, the full
solves take tens of minutes on 8 cores and are run once, here, in the CPU container) and a prefix
for config 5 (K = N = 512, ~270 k passes); one extra component is run so that the separation of
component K_s - 1 from its successor is known.

Output: tests/golden/oracle_<cfg>_<algo>.npz with
    lam      (K_s + 1,) float64   lambda_k
    iters    (K_s + 1,) int32     inner passes
    P        (N, K_s + 1) float32 loadings (unit columns)
    rows     (S,) int64           sampled row indices (np.linspace over [0, M-1])
    T_rows   (S, K_s + 1) float32 the scores at those rows
    x_fro2   float64              ||X_c||_F^2 of the centred input the oracle saw
    x_idx    (64,) int64          flat column-major indices into the RAW (uncentred) float32 input
    x_val    (64,) float32        the raw input at those indices: the tests assert that the regenerated
                                  input still IS the matrix the oracle saw (inputs.py draws U, V with a
                                  LAPACK QR; a different LAPACK could rotate the basis silently)
    meta     json string          config, K_s, seed, eps, max_iter, wall seconds, this command
The GPU parity tests (tests/test_gpu_parity.py) regenerate the same seeded input, run the CUDA
path at full size and compare against these values (tolerances of BASELINE.json's north_star).
"""
from __future__ import annotations

import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_0811_1081_b200 import inputs  # noqa: E402

# components of the full-size solve that are stored (K_s); the run itself does K_s + 1
PREFIX = {0: 8, 1: 32, 2: 64, 3: 128, 4: 16}
X_SAMPLES = 64
SAMPLED_ROWS = 256


def out_path(cfg, algo) -> str:
    return os.path.join(HERE, f"oracle_{cfg.name}_{'gs' if algo == inputs.ALGO_GS else 'nipals'}.npz")


def make(ci: int) -> None:
    cfg = inputs.config(ci)
    ks = min(PREFIX[ci], cfg.K)
    krun = min(ks + 1, cfg.N)
    t0 = time.time()
    pr = inputs.generate(cfg)
    x_idx = np.unique(np.linspace(0, cfg.M * cfg.N - 1, X_SAMPLES).astype(np.int64))
    x_val = pr.X.ravel(order="K")[x_idx].copy()                      # pr.X is Fortran-ordered: memory order = column-major
    assert pr.X.flags.f_contiguous
    Xc = oracle.center(pr.X)
    del pr
    x_fro2 = float(np.sum(Xc * Xc))
    rows = np.unique(np.linspace(0, cfg.M - 1, SAMPLED_ROWS).astype(np.int64))
    for algo in cfg.algos:
        t1 = time.time()
        r = oracle.pca(Xc, krun, cfg.eps, cfg.max_iter, algo, want_residual=False)
        wall = time.time() - t1
        meta = dict(cfg=cfg.name, M=cfg.M, N=cfg.N, K=cfg.K, K_stored=ks, K_run=krun, algo=int(algo),
                    eps=cfg.eps, max_iter=cfg.max_iter, seed=cfg.seed, oracle_wall_s=round(wall, 1),
                    threads=oracle.num_threads(),
                    command=f"python tests/golden/make_oracle_prefix.py {ci}")
        np.savez_compressed(out_path(cfg, algo), lam=r.lam, iters=r.iters, P=r.P.astype(np.float32),
                            rows=rows, T_rows=r.T[rows, :].astype(np.float32), x_fro2=np.float64(x_fro2),
                            x_idx=x_idx, x_val=x_val, meta=json.dumps(meta))
        print(f"{cfg.name} algo {algo}: K_run {krun} iters {r.iters.tolist()} lam[:4] {r.lam[:4]} "
              f"oracle {wall:.1f}s (gen+centre {t1 - t0:.1f}s)", flush=True)


if __name__ == "__main__":
    which = [int(a) for a in sys.argv[1:]] or list(range(len(inputs.CONFIGS)))
    for ci in which:
        make(ci)
