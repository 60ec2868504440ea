"""Host logic of the row-sharded multi-GPU solve (paper_0811_1081_b200/sharded.py) on CPU:
world_size 2, gloo.  The CUDA shard is replaced by a numpy stand-in with the same seven steps and the same two exchange
buffers (test infrastructure: plain fp64 numpy, the single-sweep algebra of csrc/pca_shard.cuh written out), so what is
tested is what the host adds -- where the ONE all-reduce per pass sits, the all-reduce of the column sums for the centring,
the polling of the convergence flag every few passes with harmless repeated steps after convergence -- and that a row-sharded
run gives the oracle's result of the unsharded matrix.
"""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


class NumpyShard:
    """Stand-in for sharded.CudaShard: one rank's rows, fp64 numpy (PAPER.md:1016-1038 in the single-sweep form)."""

    def __init__(self, X_local, K, eps, max_iter, algo):
        self.X = np.array(X_local, dtype=np.float64)
        self.Ml, self.N = self.X.shape
        self.K, self.eps, self.max_iter, self.gs = K, eps, max_iter, algo == 1
        L = self.N + 2 + K
        self.send = torch.zeros(L, dtype=torch.float64)
        self.recv = torch.zeros(L, dtype=torch.float64)
        self.steps_after_done = 0

    def colsums(self):
        return torch.from_numpy(self.X.sum(axis=0))

    def center(self, sums, M_total):
        self.X -= sums.numpy()[None, :] / M_total

    def begin(self):
        N, K = self.N, self.K
        self.R = self.X.copy()
        self.V = np.zeros((self.Ml, K)); self.T = np.zeros((self.Ml, K)); self.P = np.zeros((N, K)); self.W = np.zeros((N, K))
        self.lam_out = np.zeros(K); self.iters = np.zeros(K, dtype=np.int32)
        self.d = np.zeros(self.Ml); self.pdef = np.zeros(N)
        self._reset()

    def _reset(self):
        self.lam = 0.0; self.it = 0; self.is_done = False; self.first = True

    def _publish(self, t, k):
        B = self.V[:, :k].T @ t if (self.gs and k > 0 and not self.first_sweep) else np.zeros(k)
        buf = np.zeros(self.N + 2 + self.K)
        buf[:self.N] = self.R.T @ t
        buf[self.N] = t @ t
        buf[self.N + 2:self.N + 2 + k] = B
        self.send.copy_(torch.from_numpy(buf))
        self.ttil = t

    def component(self, k):
        self.R -= np.outer(self.d, self.pdef)                        # pending deflation (S9)
        self.first_sweep = True
        self._publish(self.R[:, k].copy(), k)                        # S1, S2

    def step(self, k):
        if self.is_done:
            self.steps_after_done += 1
            return
        r = self.recv.numpy()
        q, s, B = r[:self.N], r[self.N], r[self.N + 2:self.N + 2 + k]
        gsk = self.gs and k > 0
        if not self.first:
            ln = np.sqrt(s - B @ B)                                  # S7
            if abs(self.lam - ln) < self.eps * ln or self.it >= self.max_iter:   # S8
                self.lam_new = ln
                self.praw = q - self.W[:, :k] @ B if gsk else q.copy()
                self.Bfin = B.copy()
                self.is_done = True
                return
            self.lam = ln
        praw = q - self.W[:, :k] @ B if (gsk and not self.first) else q.copy()
        ph = praw - self.P[:, :k] @ (self.P[:, :k].T @ praw) if gsk else praw    # S3
        self.p = ph / np.linalg.norm(ph)                             # S4
        self.first = False
        self.it += 1
        self.first_sweep = False
        self._publish(self.R @ self.p, k)                            # S5 (+ S2 of the next pass, S6)

    def done(self):
        return int(self.is_done)

    def finish(self, k):
        t = self.ttil - self.V[:, :k] @ self.Bfin if (self.gs and k > 0) else self.ttil
        lam = self.lam_new
        self.d = t.copy(); self.pdef = self.p.copy()
        self.T[:, k] = t
        self.V[:, k] = t / lam
        self.P[:, k] = self.p
        self.W[:, k] = self.praw / lam - lam * self.p
        self.lam_out[k] = lam; self.iters[k] = self.it
        self._reset()

    def end(self, want_residual=False):
        out = dict(T=self.T, P=self.P, lam=self.lam_out, iters=self.iters, steps_after_done=self.steps_after_done)
        if want_residual:
            out["R"] = self.R - np.outer(self.d, self.pdef)
        return out


def _problem():
    from paper_0811_1081_b200 import inputs
    cfg = inputs.scaled(inputs.config(1), 300, 40, K=5)
    return cfg, inputs.generate(cfg).X.astype(np.float64)


def _worker(rank, world, port, out, algo):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_0811_1081_b200 import sharded
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg, X = _problem()
    cut = 170                                                        # uneven split: 170 + 130 rows
    Xl = X[:cut] if rank == 0 else X[cut:]
    res = sharded.solve_sharded([NumpyShard(Xl, cfg.K, 1e-10, 500, algo)], X.shape[0], cfg.K, check_every=3, want_residual=True)[0]
    out[rank] = {k: (v if not isinstance(v, np.ndarray) else v.copy()) for k, v in res.items()}
    dist.barrier()
    dist.destroy_process_group()


def _run(algo, port):
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(2, port, out, algo), nprocs=2, join=True)
        return dict(out)


def test_sharded_host_logic_gloo_world2_matches_the_oracle():
    import oracle
    cfg, X = _problem()
    Xc = X - X.mean(axis=0, keepdims=True)
    for algo, port in ((1, 29541), (0, 29542)):
        res = _run(algo, port)
        ref = oracle.pca(np.asfortranarray(Xc), cfg.K, 1e-10, 500, algo, want_residual=True)
        r0, r1 = res[0], res[1]
        np.testing.assert_array_equal(r0["P"], r1["P"])              # replicated loads side: identical on both ranks
        np.testing.assert_array_equal(r0["lam"], r1["lam"])
        np.testing.assert_array_equal(r0["iters"], r1["iters"])
        assert r0["iters"].tolist() == ref.iters[:cfg.K].tolist()
        np.testing.assert_allclose(r0["lam"], ref.lam[:cfg.K], rtol=1e-10)
        T = np.vstack([r0["T"], r1["T"]])
        R = np.vstack([r0["R"], r1["R"]])
        np.testing.assert_allclose(r0["P"], ref.P[:, :cfg.K], atol=1e-8)
        np.testing.assert_allclose(T, ref.T[:, :cfg.K], atol=1e-8 * np.max(np.abs(ref.T)))
        np.testing.assert_allclose(R, ref.R, atol=1e-8 * np.max(np.abs(Xc)))
        assert r0["steps_after_done"] > 0                            # the flag is polled every 3 passes: repeats did happen
        assert r0["exchanges"] % 3 == 0 and r0["exchanges"] >= int(ref.iters[:cfg.K].sum()) + cfg.K
