"""GPU test of the no-allocation entry point pca_run_small_static (include/pca.h; paper_0811_1081_b200/csrc/pca_noalloc.cu).

The entry point runs the one-CTA solve kernel with its scratch (the row-major working copy of the residual) in a static
device array of the library instead of a caller-owned workspace.  Its output is compared with the existing path -- pca_run on
PCA_OPT_PATH = 6, same centred input -- on two calls in a row that share the array (different shapes, no synchronisation in
between), within the tolerances of the parity tests (parity_util: TOL_LAMBDA, TOL_COS); since both run the same kernel on the
same input the results are in fact expected to be identical, which is asserted as well.

The file name sorts last so that `pytest -x` collects it after every other test.
"""
import numpy as np
import pytest

from paper_0811_1081_b200 import inputs

from parity_util import TOL_COS, TOL_LAMBDA, f64, signed_cos

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (the library has no CPU fallback)")
    from paper_0811_1081_b200 import binding as b
    b.load_library()
    return b


# (config index, M, N, K, algo): shapes of the one-CTA kernel -- GT = 8 / 16 / 64 threads per row, ragged M and N, K = N
CASES = {
    "cfg1_gs": (0, 256, 64, 8, inputs.ALGO_GS),
    "cfg1_nipals": (0, 256, 64, 8, inputs.ALGO_NIPALS),
    "ragged": (4, 101, 37, 5, inputs.ALGO_GS),
    "wide": (4, 50, 300, 10, inputs.ALGO_GS),
    "full_rank": (0, 200, 24, 24, inputs.ALGO_GS),
    "max_rows": (0, 448, 64, 6, inputs.ALGO_GS),
}


def _problem(name):
    ci, M, N, K, algo = CASES[name]
    cfg = inputs.scaled(inputs.config(ci), M, N, K)
    return cfg, inputs.generate(cfg).X, algo


def _existing_path(binding, name):
    cfg, X, algo = _problem(name)
    ref = binding.fit(X, cfg.K, cfg.eps, cfg.max_iter, algo, path=binding.PCA_PATH_ONE_CTA, want_residual=True)
    assert ref["info"]["path"] == "single-sweep one-CTA"
    return cfg, algo, ref


class _StaticCall:
    """Device buffers of one pca_run_small_static call, allocated up front (the call itself allocates nothing)."""

    def __init__(self, binding, cfg, algo, Xc_np):
        import torch
        self.cfg, self.algo = cfg, algo
        self.X = binding.from_colmajor(Xc_np)                       # the centred matrix the existing path solved
        self.T = torch.full((cfg.K, cfg.M), float("nan"), dtype=torch.float32, device="cuda")
        self.P = torch.full((cfg.K, cfg.N), float("nan"), dtype=torch.float32, device="cuda")
        self.lam = torch.full((cfg.K,), float("nan"), dtype=torch.float32, device="cuda")
        self.iters = torch.full((cfg.K,), -1, dtype=torch.int32, device="cuda")
        self.R = torch.full((cfg.N, cfg.M), float("nan"), dtype=torch.float32, device="cuda")

    def enqueue(self, binding):
        binding.pca_run_small_static(self.X, self.T, self.P, self.lam, self.iters, eps=self.cfg.eps,
                                     max_iter=self.cfg.max_iter, algo=self.algo, R=self.R)

    def results(self, binding):
        return dict(T=binding.to_colmajor(self.T), P=binding.to_colmajor(self.P), lam=self.lam.cpu().numpy(),
                    iters=self.iters.cpu().numpy(), R=binding.to_colmajor(self.R))


def _assert_matches(got, ref, what):
    K = len(ref["lam"])
    lam_ref = f64(ref["lam"])
    scale = max(float(lam_ref.max()), 1e-30)
    # the tolerances of the parity tests ...
    np.testing.assert_array_equal(got["iters"], ref["iters"], err_msg=what)
    assert np.max(np.abs(f64(got["lam"]) - lam_ref)) <= TOL_LAMBDA * scale, what
    for k in range(K):
        if ref["lam"][k] > 0:
            assert signed_cos(got["P"][:, k], ref["P"][:, k]) >= 1.0 - TOL_COS, (what, k)
            assert signed_cos(got["T"][:, k], ref["T"][:, k]) >= 1.0 - TOL_COS, (what, k)
    assert np.max(np.abs(f64(got["R"]) - f64(ref["R"]))) <= TOL_LAMBDA * scale, what
    # ... and, the same kernel on the same input: identical
    for key in ("lam", "T", "P", "R"):
        np.testing.assert_array_equal(got[key], ref[key], err_msg=f"{what}: {key}")


@pytest.mark.parametrize("first,second", [("cfg1_gs", "wide"), ("ragged", "cfg1_nipals"), ("max_rows", "full_rank")])
def test_two_calls_in_a_row_match_the_existing_path(binding, first, second):
    import torch
    refs = [_existing_path(binding, n) for n in (first, second)]
    calls = [_StaticCall(binding, cfg, algo, ref["Xc"]) for cfg, algo, ref in refs]
    torch.cuda.synchronize()
    for c in calls:                    # back to back on one stream: the second call reuses the array the first one filled
        c.enqueue(binding)
    torch.cuda.synchronize()
    for name, c, (_, _, ref) in zip((first, second), calls, refs):
        _assert_matches(c.results(binding), ref, name)


def test_same_problem_twice_and_no_device_allocation(binding):
    import torch
    cfg, algo, ref = _existing_path(binding, "cfg1_gs")
    a = _StaticCall(binding, cfg, algo, ref["Xc"])
    b = _StaticCall(binding, cfg, algo, ref["Xc"])
    a.enqueue(binding)                 # (the first call on a device also does the one-time set-up)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    reserved0 = torch.cuda.memory_reserved()
    b.enqueue(binding)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_reserved() == reserved0
    assert free1 >= free0, "pca_run_small_static must not allocate device memory"
    ra, rb = a.results(binding), b.results(binding)
    _assert_matches(ra, ref, "first call")
    _assert_matches(rb, ref, "second call")


def test_residual_is_optional(binding):
    import torch
    cfg, algo, ref = _existing_path(binding, "ragged")
    c = _StaticCall(binding, cfg, algo, ref["Xc"])
    binding.pca_run_small_static(c.X, c.T, c.P, c.lam, c.iters, eps=cfg.eps, max_iter=cfg.max_iter, algo=algo, R=None)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(c.lam.cpu().numpy(), ref["lam"])
    np.testing.assert_array_equal(binding.to_colmajor(c.P), ref["P"])
    assert bool(torch.isnan(c.R).all())


@pytest.mark.parametrize("M,N,K", [(449, 64, 4), (225, 128, 4), (57, 512, 4), (64, 513, 4), (4096, 1024, 8)])
def test_sizes_beyond_the_static_scratch_are_rejected(binding, M, N, K):
    import torch
    assert binding.pca_small_static_scratch_bytes() == 114688
    X = torch.zeros((N, M), dtype=torch.float32, device="cuda")
    T = torch.zeros((K, M), dtype=torch.float32, device="cuda")
    P = torch.zeros((K, N), dtype=torch.float32, device="cuda")
    lam = torch.zeros(K, dtype=torch.float32, device="cuda")
    iters = torch.zeros(K, dtype=torch.int32, device="cuda")
    with pytest.raises(binding.PcaError) as ei:
        binding.pca_run_small_static(X, T, P, lam, iters)
    assert ei.value.code == binding.PCA_EUNSUPPORTED
    msg = str(ei.value)
    assert ("static scratch" in msg and "114688" in msg) or "maximum of 512 columns" in msg, msg


def test_bad_arguments_are_rejected(binding):
    import torch
    X = torch.zeros((8, 32), dtype=torch.float32, device="cuda")
    T = torch.zeros((9, 32), dtype=torch.float32, device="cuda")       # K = 9 > N = 8
    P = torch.zeros((9, 8), dtype=torch.float32, device="cuda")
    lam = torch.zeros(9, dtype=torch.float32, device="cuda")
    iters = torch.zeros(9, dtype=torch.int32, device="cuda")
    with pytest.raises(binding.PcaError) as ei:
        binding.pca_run_small_static(X, T, P, lam, iters)
    assert ei.value.code == binding.PCA_EINVAL


def test_can_be_captured_into_a_cuda_graph(binding):
    """What the entry point is for: enqueued under stream capture (where cudaMalloc is not allowed), replayed twice."""
    import torch
    cfg, algo, ref = _existing_path(binding, "cfg1_gs")
    c = _StaticCall(binding, cfg, algo, ref["Xc"])
    c.enqueue(binding)                 # one-time set-up of the device outside the capture
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        c.enqueue(binding)
    for _ in range(2):
        c.lam.zero_()
        c.P.zero_()
        graph.replay()
        torch.cuda.synchronize()
        _assert_matches(c.results(binding), ref, "graph replay")
