"""Thin Python binding of the C ABI in include/pca.h (argument marshalling only).

Every function has the name of the C entry point it calls; every step of the path runs in the
CUDA kernels of libpca_b200.so.  torch is used only for device memory and streams.  There is no
CPU fallback: if the library is missing it is built (nvcc), and if there is no CUDA device
`pca_create` fails with PCA_ECUDA -> PcaError.

Matrix layout: an M x N column-major matrix (ld = M) is a contiguous torch tensor
of shape (N, M); helpers `from_colmajor` / `to_colmajor` convert from/to numpy (M, N) arrays.
"""
from __future__ import annotations

import ctypes
import os

PCA_ALGO_NIPALS = 0
PCA_ALGO_GS = 1

PCA_OK, PCA_EINVAL, PCA_EALIGN, PCA_ECUDA, PCA_EWORKSPACE, PCA_EUNSUPPORTED, PCA_EPROTOCOL = range(7)

PCA_OPT_PATH, PCA_OPT_CTAS, PCA_OPT_CENTER_MODE, PCA_OPT_TRACE, PCA_OPT_OWNERS, PCA_OPT_KDIRECT, PCA_OPT_TEST_MODE = 1, 2, 3, 4, 5, 6, 7
PCA_OPT_STAGNATION, PCA_OPT_OUTPUT, PCA_OPT_GS_PASSES, PCA_OPT_RING_ROWS, PCA_OPT_RING_SLOTS = 8, 9, 10, 11, 12
PCA_OPT_STORAGE = 14
PCA_OPT_DEFER_S3 = 15
PCA_PATH_F64 = 8
(PCA_PATH_AUTO, PCA_PATH_STREAMING, PCA_PATH_RESIDENT, PCA_PATH_FUSED_STREAMING, PCA_PATH_FUSED_RESIDENT,
 PCA_PATH_REGISTER, PCA_PATH_ONE_CTA, PCA_PATH_TMA_STREAMING) = 0, 1, 2, 3, 4, 5, 6, 7
(PCA_INFO_PATH, PCA_INFO_CTAS, PCA_INFO_THREADS, PCA_INFO_SMEM_BYTES, PCA_INFO_ROWS_PER_CTA,
 PCA_INFO_LAUNCHES_PER_RUN, PCA_INFO_NUM_SMS, PCA_INFO_ROW_GROUP_THREADS, PCA_INFO_RUN_STATUS, PCA_INFO_OWNERS,
 PCA_INFO_RING_ROWS, PCA_INFO_RING_SLOTS) = range(1, 13)

EXPORTED_SYMBOLS = (
    "pca_create", "pca_set_option", "pca_get_info", "pca_workspace_bytes", "pca_set_workspace",
    "pca_center", "pca_run", "pca_residual", "pca_fit_host", "pca_destroy", "pca_strerror",
    "pca_last_cuda_error", "pca_trace", "pca_center_f64", "pca_run_f64", "pca_residual_f64",
    "pca_shard_create", "pca_shard_workspace_bytes", "pca_shard_set_workspace", "pca_shard_exchange", "pca_shard_colsums",
    "pca_shard_center", "pca_shard_begin", "pca_shard_component", "pca_shard_pass", "pca_shard_done", "pca_shard_finish_component",
    "pca_shard_end", "pca_shard_destroy", "pca_shard_last_cuda_error",
    "pca_run_small_static", "pca_small_static_scratch_bytes", "pca_small_static_last_error", "pca_small_static_last_cuda_error",
)

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpca_b200.so")


class PcaError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        super().__init__(f"{where}: {detail or code}")


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libpca_b200.so (building it with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    path = _build.build()
    lib = ctypes.CDLL(path)
    vp, i64, i32, f64 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
    lib.pca_create.argtypes = [ctypes.POINTER(vp), i64, i64, i32, f64, i32, i32]
    lib.pca_create.restype = i32
    lib.pca_set_option.argtypes = [vp, i32, i64]
    lib.pca_get_info.argtypes = [vp, i32, ctypes.POINTER(i64)]
    lib.pca_workspace_bytes.argtypes = [vp]
    lib.pca_workspace_bytes.restype = ctypes.c_size_t
    lib.pca_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
    lib.pca_center.argtypes = [vp, vp, vp]
    lib.pca_run.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.pca_residual.argtypes = [vp, ctypes.POINTER(vp)]
    lib.pca_fit_host.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.pca_destroy.argtypes = [vp]
    lib.pca_destroy.restype = None
    lib.pca_strerror.argtypes = [i32]
    lib.pca_strerror.restype = ctypes.c_char_p
    lib.pca_last_cuda_error.argtypes = [vp]
    lib.pca_trace.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(i64)]
    lib.pca_center_f64.argtypes = [vp, vp, vp]
    lib.pca_run_f64.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.pca_residual_f64.argtypes = [vp, ctypes.POINTER(vp)]
    lib.pca_shard_create.argtypes = [ctypes.POINTER(vp), i64, i64, i32, f64, i32, i32]
    lib.pca_shard_workspace_bytes.argtypes = [vp]
    lib.pca_shard_workspace_bytes.restype = ctypes.c_size_t
    lib.pca_shard_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
    lib.pca_shard_exchange.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(i64)]
    lib.pca_shard_colsums.argtypes = [vp, vp, vp, vp]
    lib.pca_shard_center.argtypes = [vp, vp, vp, i64, vp]
    lib.pca_shard_begin.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.pca_shard_component.argtypes = [vp, i32, vp]
    lib.pca_shard_pass.argtypes = [vp, i32, vp]
    lib.pca_shard_done.argtypes = [vp, ctypes.POINTER(i32), vp]
    lib.pca_shard_finish_component.argtypes = [vp, i32, vp]
    lib.pca_shard_end.argtypes = [vp, vp, vp]
    lib.pca_shard_destroy.argtypes = [vp]
    lib.pca_shard_destroy.restype = None
    lib.pca_shard_last_cuda_error.argtypes = [vp]
    lib.pca_run_small_static.argtypes = [vp, i64, i64, i32, f64, i32, i32, vp, vp, vp, vp, vp, vp]
    lib.pca_small_static_scratch_bytes.argtypes = []
    lib.pca_small_static_scratch_bytes.restype = ctypes.c_size_t
    lib.pca_small_static_last_error.argtypes = []
    lib.pca_small_static_last_error.restype = ctypes.c_char_p
    lib.pca_small_static_last_cuda_error.argtypes = []
    _lib = lib
    return lib


def pca_strerror(code: int) -> str:
    return load_library().pca_strerror(int(code)).decode()


def _check(code: int, where: str, ctx=None):
    if code != PCA_OK:
        detail = pca_strerror(code)
        if ctx is not None and code == PCA_ECUDA:
            detail += f" (cudaError {load_library().pca_last_cuda_error(ctx)})"
        raise PcaError(code, where, detail)


def _stream_ptr(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


class PcaContext:
    """Owns a pca_ctx* and (optionally) the torch workspace tensor handed to it."""

    def __init__(self, M: int, N: int, K: int, eps: float = 1e-7, max_iter: int = 10000,
                 algo: int = PCA_ALGO_GS):
        self._lib = load_library()
        self._ctx = ctypes.c_void_p()
        self.M, self.N, self.K, self.eps, self.max_iter, self.algo = int(M), int(N), int(K), float(eps), int(max_iter), int(algo)
        self._ws = None
        _check(self._lib.pca_create(ctypes.byref(self._ctx), self.M, self.N, self.K, self.eps,
                                    self.max_iter, self.algo), "pca_create")

    # -- plan ---------------------------------------------------------------------------------
    def pca_set_option(self, option: int, value: int) -> None:
        _check(self._lib.pca_set_option(self._ctx, int(option), int(value)), "pca_set_option", self._ctx)
        self._ws = None

    def pca_get_info(self, field: int) -> int:
        v = ctypes.c_int64()
        _check(self._lib.pca_get_info(self._ctx, int(field), ctypes.byref(v)), "pca_get_info")
        return int(v.value)

    def info(self) -> dict:
        return {
            "path": {1: "two-sweep streaming", 2: "two-sweep resident", 3: "single-sweep streaming",
                     4: "single-sweep resident",
                     5: "single-sweep register-resident", 6: "single-sweep one-CTA",
                     7: "single-sweep streaming (TMA ring)", 8: "two-sweep streaming fp64"}.get(self.pca_get_info(PCA_INFO_PATH), "?"),
            "ctas": self.pca_get_info(PCA_INFO_CTAS),
            "threads": self.pca_get_info(PCA_INFO_THREADS),
            "smem_bytes": self.pca_get_info(PCA_INFO_SMEM_BYTES),
            "rows_per_cta": self.pca_get_info(PCA_INFO_ROWS_PER_CTA),
            "launches_per_run": self.pca_get_info(PCA_INFO_LAUNCHES_PER_RUN),
            "num_sms": self.pca_get_info(PCA_INFO_NUM_SMS),
            "row_group_threads": self.pca_get_info(PCA_INFO_ROW_GROUP_THREADS),
            "owners": self.pca_get_info(PCA_INFO_OWNERS),
            "ring_rows": self.pca_get_info(PCA_INFO_RING_ROWS),
            "ring_slots": self.pca_get_info(PCA_INFO_RING_SLOTS),
        }

    def pca_workspace_bytes(self) -> int:
        return int(self._lib.pca_workspace_bytes(self._ctx))

    def pca_set_workspace(self, ws_tensor) -> None:
        nbytes = ws_tensor.numel() * ws_tensor.element_size()
        _check(self._lib.pca_set_workspace(self._ctx, ctypes.c_void_p(ws_tensor.data_ptr()), nbytes),
               "pca_set_workspace")
        self._ws = ws_tensor

    def ensure_workspace(self, device="cuda"):
        import torch
        if self._ws is None:
            ws = torch.empty(self.pca_workspace_bytes() + 256, dtype=torch.uint8, device=device)
            off = (-ws.data_ptr()) % 256
            self.pca_set_workspace(ws[off:off + self.pca_workspace_bytes()])
            self._ws_base = ws
        return self._ws

    # -- the path -----------------------------------------------------------------------------
    def pca_center(self, X, stream=None) -> None:
        """X: torch float32 CUDA tensor of shape (N, M) (= M x N column-major), centred in place."""
        self._check_mat(X, self.N, self.M, "X")
        _check(self._lib.pca_center(self._ctx, ctypes.c_void_p(X.data_ptr()), _stream_ptr(stream)),
               "pca_center", self._ctx)

    def pca_run(self, X, T, P, lam, iters, stream=None) -> None:
        """X (N,M), T (K,M), P (K,N) float32; lam (K,) float32; iters (K,) int32 -- all CUDA, contiguous."""
        import torch
        self._check_mat(X, self.N, self.M, "X")
        self._check_mat(T, self.K, self.M, "T")
        self._check_mat(P, self.K, self.N, "P")
        if lam.dtype != torch.float32 or lam.numel() != self.K or not lam.is_cuda or not lam.is_contiguous():
            raise ValueError("lambda must be a contiguous CUDA float32 tensor of K elements")
        if iters.dtype != torch.int32 or iters.numel() != self.K or not iters.is_cuda or not iters.is_contiguous():
            raise ValueError("iters must be a contiguous CUDA int32 tensor of K elements")
        self.ensure_workspace(X.device)
        vp = ctypes.c_void_p
        _check(self._lib.pca_run(self._ctx, vp(X.data_ptr()), vp(T.data_ptr()), vp(P.data_ptr()),
                                 vp(lam.data_ptr()), vp(iters.data_ptr()), _stream_ptr(stream)),
               "pca_run", self._ctx)

    # -- fp64 storage (PCA_OPT_STORAGE = 1): same calls on float64 tensors ----------------------
    def pca_center_f64(self, X, stream=None) -> None:
        self._check_mat(X, self.N, self.M, "X", f64=True)
        _check(self._lib.pca_center_f64(self._ctx, ctypes.c_void_p(X.data_ptr()), _stream_ptr(stream)), "pca_center_f64", self._ctx)

    def pca_run_f64(self, X, T, P, lam, iters, stream=None) -> None:
        import torch
        self._check_mat(X, self.N, self.M, "X", f64=True)
        self._check_mat(T, self.K, self.M, "T", f64=True)
        self._check_mat(P, self.K, self.N, "P", f64=True)
        if lam.dtype != torch.float64 or lam.numel() != self.K or not lam.is_cuda or not lam.is_contiguous():
            raise ValueError("lambda must be a contiguous CUDA float64 tensor of K elements")
        if iters.dtype != torch.int32 or iters.numel() != self.K or not iters.is_cuda or not iters.is_contiguous():
            raise ValueError("iters must be a contiguous CUDA int32 tensor of K elements")
        self.ensure_workspace(X.device)
        vp = ctypes.c_void_p
        _check(self._lib.pca_run_f64(self._ctx, vp(X.data_ptr()), vp(T.data_ptr()), vp(P.data_ptr()),
                                     vp(lam.data_ptr()), vp(iters.data_ptr()), _stream_ptr(stream)), "pca_run_f64", self._ctx)

    def pca_residual_f64(self):
        import torch
        ptr = ctypes.c_void_p()
        _check(self._lib.pca_residual_f64(self._ctx, ctypes.byref(ptr)), "pca_residual_f64")
        off = ptr.value - self._ws.data_ptr()
        return self._ws[off:off + self.M * self.N * 8].view(torch.float64).view(self.N, self.M)

    def pca_residual(self):
        """View of the residual R inside the workspace as a (N, M) torch tensor (valid after pca_run)."""
        import torch
        ptr = ctypes.c_void_p()
        _check(self._lib.pca_residual(self._ctx, ctypes.byref(ptr)), "pca_residual")
        off = ptr.value - self._ws.data_ptr()
        nbytes = self.M * self.N * 4
        return self._ws[off:off + nbytes].view(torch.float32).view(self.N, self.M)

    def pca_trace(self):
        """Phase trace of the last pca_run as a (n, 2) int64 numpy array of (phase id, SM cycle counter)."""
        import numpy as np
        import torch
        ptr, cap = ctypes.c_void_p(), ctypes.c_int64()
        _check(self._lib.pca_trace(self._ctx, ctypes.byref(ptr), ctypes.byref(cap)), "pca_trace")
        off = ptr.value - self._ws.data_ptr()
        rec = self._ws[off:off + 8 * (cap.value + 1)].view(torch.int64).cpu().numpy()
        n = int(rec[0])
        body = rec[1:1 + n]
        return np.stack([(body >> 56) & 0xff, body & ((1 << 56) - 1)], axis=1)

    def pca_fit_host(self, X_host, T_host, P_host, lam_host, iters_host, stream=None) -> None:
        """Host (CPU, ideally pinned) torch tensors: X (N,M) NOT centred in; T (K,M), P (K,N), lam, iters out."""
        vp = ctypes.c_void_p
        for t in (X_host, T_host, P_host, lam_host, iters_host):
            if t.is_cuda or not t.is_contiguous():
                raise ValueError("pca_fit_host takes contiguous host tensors")
        _check(self._lib.pca_fit_host(self._ctx, vp(X_host.data_ptr()), vp(T_host.data_ptr()),
                                      vp(P_host.data_ptr()), vp(lam_host.data_ptr()),
                                      vp(iters_host.data_ptr()), _stream_ptr(stream)),
               "pca_fit_host", self._ctx)

    # -- misc ---------------------------------------------------------------------------------
    @staticmethod
    def _check_mat(t, rows, cols, name, f64=False):
        import torch
        want = torch.float64 if f64 else torch.float32
        if (not t.is_cuda) or t.dtype != want or tuple(t.shape) != (rows, cols) or not t.is_contiguous():
            raise ValueError(f"{name} must be a contiguous CUDA {want} tensor of shape ({rows}, {cols})")

    def pca_destroy(self) -> None:
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self._lib.pca_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.pca_destroy()
        except Exception:
            pass


# ---- no-allocation entry point (include/pca.h: pca_run_small_static) -----------------------------------
def pca_small_static_scratch_bytes() -> int:
    return int(load_library().pca_small_static_scratch_bytes())


def pca_run_small_static(X, T, P, lam, iters, eps=1e-7, max_iter=10000, algo=PCA_ALGO_GS, R=None, stream=None) -> None:
    """X (N,M) centred, T (K,M), P (K,N) float32; lam (K,) float32; iters (K,) int32; R (N,M) float32 or None -- CUDA,
    contiguous.  Only enqueues kernels; allocates nothing (the scratch is a static device array of the library)."""
    import torch
    lib = load_library()
    N, M = X.shape
    K = T.shape[0]
    PcaContext._check_mat(X, N, M, "X")
    PcaContext._check_mat(T, K, M, "T")
    PcaContext._check_mat(P, K, N, "P")
    if R is not None:
        PcaContext._check_mat(R, N, M, "R")
    if lam.dtype != torch.float32 or lam.numel() != K or not lam.is_cuda or not lam.is_contiguous():
        raise ValueError("lambda must be a contiguous CUDA float32 tensor of K elements")
    if iters.dtype != torch.int32 or iters.numel() != K or not iters.is_cuda or not iters.is_contiguous():
        raise ValueError("iters must be a contiguous CUDA int32 tensor of K elements")
    vp = ctypes.c_void_p
    code = lib.pca_run_small_static(vp(X.data_ptr()), M, N, K, float(eps), int(max_iter), int(algo), vp(T.data_ptr()),
                                    vp(P.data_ptr()), vp(lam.data_ptr()), vp(iters.data_ptr()),
                                    vp(R.data_ptr()) if R is not None else vp(), _stream_ptr(stream))
    if code != PCA_OK:
        raise PcaError(code, "pca_run_small_static", lib.pca_small_static_last_error().decode() or pca_strerror(code))


# ---- numpy <-> torch layout helpers (no arithmetic) ---------------------------------------------
def from_colmajor(X_np, device="cuda"):
    """numpy (M, N) array (any order) -> torch (N, M) contiguous float32 tensor on `device`."""
    import numpy as np
    import torch
    return torch.from_numpy(np.ascontiguousarray(np.asarray(X_np, dtype=np.float32).T)).to(device)


def to_colmajor(t):
    """torch (N, M) tensor -> numpy (M, N) Fortran-ordered array."""
    return t.detach().cpu().numpy().T


def fit(X_np, K, eps=1e-7, max_iter=10000, algo=PCA_ALGO_GS, center=True, path=PCA_PATH_AUTO, ctas=0,
        want_residual=False, test_mode=0, options=None):
    """One-call helper used by tests / smoke: numpy (M, N) float32 in -> dict of numpy results.

    Runs pca_center (optional) and pca_run on the GPU through the C ABI."""
    import torch
    M, N = X_np.shape
    ctx = PcaContext(M, N, K, eps, max_iter, algo)
    if path != PCA_PATH_AUTO:
        ctx.pca_set_option(PCA_OPT_PATH, path)
    if ctas:
        ctx.pca_set_option(PCA_OPT_CTAS, ctas)
    if test_mode:
        ctx.pca_set_option(PCA_OPT_TEST_MODE, test_mode)
    for opt, val in (options or {}).items():
        ctx.pca_set_option(opt, val)
    X = from_colmajor(X_np)
    if center:
        ctx.pca_center(X)
    T = torch.empty((K, M), dtype=torch.float32, device="cuda")
    P = torch.empty((K, N), dtype=torch.float32, device="cuda")
    lam = torch.empty(K, dtype=torch.float32, device="cuda")
    iters = torch.empty(K, dtype=torch.int32, device="cuda")
    ctx.pca_run(X, T, P, lam, iters)
    torch.cuda.synchronize()
    if ctx.pca_get_info(PCA_INFO_RUN_STATUS) != 0:
        raise PcaError(PCA_EPROTOCOL, "pca_run", "a cross-CTA exchange wait gave up (PCA_INFO_RUN_STATUS != 0)")
    out = dict(T=to_colmajor(T), P=to_colmajor(P), lam=lam.cpu().numpy(), iters=iters.cpu().numpy(),
               Xc=to_colmajor(X), info=ctx.info())
    if want_residual:
        out["R"] = to_colmajor(ctx.pca_residual()).copy()
    ctx.pca_destroy()
    return out


def fit_f64(X_np, K, eps=1e-7, max_iter=10000, algo=PCA_ALGO_GS, center=True, ctas=0, want_residual=False, options=None):
    """fp64-storage sibling of fit(): numpy (M, N) float64 in -> dict of float64 numpy results (PCA_OPT_STORAGE = 1)."""
    import numpy as np
    import torch
    M, N = X_np.shape
    ctx = PcaContext(M, N, K, eps, max_iter, algo)
    ctx.pca_set_option(PCA_OPT_STORAGE, 1)
    if ctas:
        ctx.pca_set_option(PCA_OPT_CTAS, ctas)
    for opt, val in (options or {}).items():
        ctx.pca_set_option(opt, val)
    X = torch.from_numpy(np.ascontiguousarray(np.asarray(X_np, dtype=np.float64).T)).cuda()
    if center:
        ctx.pca_center_f64(X)
    T = torch.empty((K, M), dtype=torch.float64, device="cuda")
    P = torch.empty((K, N), dtype=torch.float64, device="cuda")
    lam = torch.empty(K, dtype=torch.float64, device="cuda")
    iters = torch.empty(K, dtype=torch.int32, device="cuda")
    ctx.pca_run_f64(X, T, P, lam, iters)
    torch.cuda.synchronize()
    out = dict(T=to_colmajor(T), P=to_colmajor(P), lam=lam.cpu().numpy(), iters=iters.cpu().numpy(), Xc=to_colmajor(X), info=ctx.info())
    if want_residual:
        out["R"] = to_colmajor(ctx.pca_residual_f64()).copy()
    ctx.pca_destroy()
    return out
