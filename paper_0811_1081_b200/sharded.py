"""Row-sharded multi-GPU solve: argument marshalling and the calling sequence of the
pca_shard_* entry points (include/pca.h).  Every step of the path runs in the library's CUDA kernels; this module only
enqueues them and places the ONE all-reduce per inner pass (torch.distributed: NCCL between GPUs, gloo in the CPU tests).

    one process per GPU:   out = solve_sharded([CudaShard(X_local, K, eps, max_iter, algo)], M_total, group=None)
    one process, G shards on one GPU (tests: the ranks emulated as sequential launches, no kernel waits on another):
                           outs = solve_sharded([CudaShard(X_g, ...) for g in range(G)], M_total)

`solve_sharded` talks to the shards through seven methods (colsums, center, begin, component, step, done, finish, end) and two
tensors (send, recv), so the host logic -- where the exchange sits, the done-flag polling, the harmless repeats after
convergence -- is tested on CPU with a stand-in shard (tests/test_sharded_host.py, world_size 2, gloo).
"""
from __future__ import annotations

import ctypes


def _exchange(shards, group, world):
    """recv <- sum over ALL shards of all ranks of send (fixed order: local shards in list order, then the all-reduce)."""
    import torch.distributed as dist
    total = shards[0].send.clone()
    for s in shards[1:]:
        total += s.send
    if world > 1:
        dist.all_reduce(total, group=group)
    for s in shards:
        s.recv.copy_(total)


def solve_sharded(shards, M_total, K, group=None, check_every=4, center=True, want_residual=False):
    """Run the sharded solve on this process's shards (usually one).  Returns the list of per-shard result dicts."""
    import torch.distributed as dist
    world = dist.get_world_size(group) if (dist.is_available() and dist.is_initialized()) else 1
    if center:                                                       # S0: column means over ALL rows
        sums = [s.colsums() for s in shards]
        total = sums[0].clone()
        for t in sums[1:]:
            total += t
        if world > 1:
            dist.all_reduce(total, group=group)
        for s in shards:
            s.center(total, M_total)
    for s in shards:
        s.begin()
    passes = 0
    for k in range(K):
        for s in shards:
            s.component(k)
        _exchange(shards, group, world)
        while True:
            for _ in range(check_every):                             # steps after convergence are no-ops on the device
                for s in shards:
                    s.step(k)
                _exchange(shards, group, world)
                passes += 1
            flags = [s.done() for s in shards]
            assert len(set(flags)) == 1, "the ranks disagree on convergence: the reduced numbers were not identical"
            if flags[0]:
                break
        for s in shards:
            s.finish(k)
    return [dict(s.end(want_residual), exchanges=passes) for s in shards]


class CudaShard:
    """One rank's rows on the current CUDA device, through the C ABI (pca_shard_*)."""

    def __init__(self, X_local_np, K, eps, max_iter, algo):
        import torch
        from . import binding
        self._b = binding
        self._lib = binding.load_library()
        self.Ml, self.N = X_local_np.shape
        self.K = K
        self._ctx = ctypes.c_void_p()
        binding._check(self._lib.pca_shard_create(ctypes.byref(self._ctx), self.Ml, self.N, K, float(eps), int(max_iter), int(algo)),
                       "pca_shard_create")
        nbytes = int(self._lib.pca_shard_workspace_bytes(self._ctx))
        self._ws_base = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        off = (-self._ws_base.data_ptr()) % 256
        self._ws = self._ws_base[off:off + nbytes]
        binding._check(self._lib.pca_shard_set_workspace(self._ctx, ctypes.c_void_p(self._ws.data_ptr()), nbytes), "pca_shard_set_workspace")
        snd, rcv, cnt = ctypes.c_void_p(), ctypes.c_void_p(), ctypes.c_int64()
        binding._check(self._lib.pca_shard_exchange(self._ctx, ctypes.byref(snd), ctypes.byref(rcv), ctypes.byref(cnt)), "pca_shard_exchange")
        so, ro = snd.value - self._ws.data_ptr(), rcv.value - self._ws.data_ptr()
        self.send = self._ws[so:so + 8 * cnt.value].view(torch.float64)
        self.recv = self._ws[ro:ro + 8 * cnt.value].view(torch.float64)
        self.X = binding.from_colmajor(X_local_np)
        self.T = torch.empty((K, self.Ml), dtype=torch.float32, device="cuda")
        self.P = torch.empty((K, self.N), dtype=torch.float32, device="cuda")
        self.lam = torch.empty(K, dtype=torch.float32, device="cuda")
        self.iters = torch.empty(K, dtype=torch.int32, device="cuda")
        self._sums = torch.empty(self.N, dtype=torch.float64, device="cuda")

    def _p(self, t):
        return ctypes.c_void_p(t.data_ptr())

    def _chk(self, code, where):
        if code == self._b.PCA_ECUDA:
            raise self._b.PcaError(code, where, f"CUDA runtime error {self._lib.pca_shard_last_cuda_error(self._ctx)}")
        self._b._check(code, where)

    def colsums(self):
        self._chk(self._lib.pca_shard_colsums(self._ctx, self._p(self.X), self._p(self._sums), None), "pca_shard_colsums")
        return self._sums

    def center(self, sums_reduced, M_total):
        self._chk(self._lib.pca_shard_center(self._ctx, self._p(self.X), self._p(sums_reduced), int(M_total), None), "pca_shard_center")

    def begin(self):
        self._chk(self._lib.pca_shard_begin(self._ctx, self._p(self.X), self._p(self.T), self._p(self.P), self._p(self.lam),
                                                 self._p(self.iters), None), "pca_shard_begin")

    def component(self, k):
        self._chk(self._lib.pca_shard_component(self._ctx, int(k), None), "pca_shard_component")

    def step(self, k):
        self._chk(self._lib.pca_shard_pass(self._ctx, int(k), None), "pca_shard_pass")

    def done(self):
        flag = ctypes.c_int(0)
        self._chk(self._lib.pca_shard_done(self._ctx, ctypes.byref(flag), None), "pca_shard_done")
        return int(flag.value)

    def finish(self, k):
        self._chk(self._lib.pca_shard_finish_component(self._ctx, int(k), None), "pca_shard_finish_component")

    def end(self, want_residual=False):
        import torch
        R = torch.empty((self.N, self.Ml), dtype=torch.float32, device="cuda") if want_residual else None
        self._chk(self._lib.pca_shard_end(self._ctx, self._p(R) if want_residual else None, None), "pca_shard_end")
        torch.cuda.synchronize()
        to = self._b.to_colmajor
        out = dict(T=to(self.T), P=to(self.P), lam=self.lam.cpu().numpy(), iters=self.iters.cpu().numpy(), Xc=to(self.X))
        if want_residual:
            out["R"] = to(R)
        self._lib.pca_shard_destroy(self._ctx)
        self._ctx = ctypes.c_void_p()
        return out
