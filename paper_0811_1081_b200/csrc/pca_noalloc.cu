// =====================================================================================
// pca_noalloc.cu -- pca_run_small_static(): the one-CTA solve (pca_one.cuh, PCA_OPT_PATH 6) for callers that cannot
// allocate device memory (code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// The one-CTA kernel needs ONE piece of scratch memory: the row-major, zero-padded working copy Rrm of the residual
// (M x ldr floats: R <- X; read once into registers, written back once after the last deflation, eq. 4
// PAPER.md:42).  Everywhere else in the library that scratch is part of a caller-owned workspace; here it is the
// file-scope device array g_small_scratch below, kSmallScratchBytes = 114688 bytes (the largest M x ldr the one-CTA
// kernel accepts: M <= (512/GT)*7 rows of ldr = 8*GT floats, i.e. at most 28672 floats whatever GT is).  Every GPU that
// loads the library holds those 112 KB until the process exits.
//
// In HOST code the array's name is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, taken once per device with that device current (small_setup).
//
// The entry point calls no cudaMalloc / cudaFree and no allocating library routine, and creates no context object.
// All calls on a device share the array; it keeps the last call's contents.  Nothing in it has to start at zero: the
// transpose-in kernel overwrites every word the solve kernel reads (the rows m < M, padding columns N <= n < ldr
// included), so no clearing pass is needed.  Calls that overlap on the GPU (two streams, two host threads) RACE on the
// array: keep them on one stream, or order them with events.
// =====================================================================================
#include "../../include/pca.h"

#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "pca_one.cuh"

namespace {

constexpr size_t kSmallScratchBytes = 114688;   // 28672 floats = max over GT of ((512/GT)*7) x (8*GT)
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_small_scratch[kSmallScratchBytes];

struct SmallDevice {
  bool ready = false;
  void* scratch = nullptr;   // DEVICE address of g_small_scratch on this device (cudaGetSymbolAddress)
  int smem_optin = 0;
};
SmallDevice g_dev[kMaxDevices];
std::mutex g_mu;

thread_local char g_err[320] = "";
thread_local int g_cuda_err = 0;

inline long long round_up(long long v, long long a) { return (v + a - 1) / a * a; }
inline long long ceil_div(long long a, long long b) { return (a + b - 1) / b; }
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int fail_cuda(cudaError_t e, const char* what) {
  g_cuda_err = (int)e;
  std::snprintf(g_err, sizeof g_err, "pca_run_small_static: %s failed: %s", what, cudaGetErrorString(e));
  return PCA_ECUDA;
}

// once per device, with that device current: the device address of the static array, the shared-memory limit, and the
// dynamic shared-memory attribute of every one-CTA kernel variant (per FUNCTION: the device maximum, as in pca_api.cu)
int small_setup(int dev, SmallDevice** out) {
  std::lock_guard<std::mutex> lock(g_mu);
  SmallDevice& d = g_dev[dev];
  if (!d.ready) {
    void* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&ptr, g_small_scratch);
    if (e != cudaSuccess) return fail_cuda(e, "cudaGetSymbolAddress");
    if (!ptr) return fail_cuda(cudaErrorInvalidSymbol, "cudaGetSymbolAddress (null address)");
    int optin = 0;
    e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return fail_cuda(e, "cudaDeviceGetAttribute");
    for (int gt : {8, 16, 32, 64})
      for (int rpt : {2, 4, 7}) {
        pca::one_kernel_t fn = pca::one_kernel_lookup(gt, rpt);
        if (!fn) continue;
        e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
        if (e != cudaSuccess) return fail_cuda(e, "cudaFuncSetAttribute");
      }
    d.scratch = ptr;
    d.smem_optin = optin;
    d.ready = true;
  }
  *out = &d;
  return PCA_OK;
}

}  // namespace

extern "C" {

size_t pca_small_static_scratch_bytes(void) { return kSmallScratchBytes; }

const char* pca_small_static_last_error(void) { return g_err; }

int pca_small_static_last_cuda_error(void) { return g_cuda_err; }

int pca_run_small_static(const float* X, int64_t M, int64_t N, int K, double eps, int max_iter, int algo, float* T, float* P,
                         float* lambda, int32_t* iters, float* R, void* stream) {
  g_err[0] = 0;
  g_cuda_err = 0;
  if (!X || !T || !P || !lambda || !iters) {
    std::snprintf(g_err, sizeof g_err, "pca_run_small_static: X, T, P, lambda and iters must not be NULL");
    return PCA_EINVAL;
  }
  if (M < 1 || N < 1 || K < 1 || K > N || !(eps >= 0.0) || max_iter < 1 || (algo != PCA_ALGO_NIPALS && algo != PCA_ALGO_GS)) {
    std::snprintf(g_err, sizeof g_err,
                  "pca_run_small_static: need M >= 1, N >= 1, 1 <= K <= N, eps >= 0, max_iter >= 1, algo 0 or 1 "
                  "(got M=%lld N=%lld K=%d eps=%g max_iter=%d algo=%d)", (long long)M, (long long)N, K, eps, max_iter, algo);
    return PCA_EINVAL;
  }
  if (!aligned16(X) || !aligned16(T) || !aligned16(P) || (R && !aligned16(R))) {
    std::snprintf(g_err, sizeof g_err, "pca_run_small_static: X, T, P and R must be 16-byte aligned");
    return PCA_EALIGN;
  }
  // ---- the plan of the one-CTA kernel (same rules as PCA_OPT_PATH = 6): GT threads share a row, RPT rows per group ----
  if (N > 512) {
    std::snprintf(g_err, sizeof g_err, "pca_run_small_static: N = %lld exceeds the maximum of 512 columns", (long long)N);
    return PCA_EUNSUPPORTED;
  }
  int GT = 8;
  while (8LL * GT < N) GT *= 2;
  const int NG = pca::kThreads / GT, ldr = 8 * GT;
  const long long max_rows = (long long)NG * 7;
  const long long need = M * (long long)ldr * 4;
  if (M > max_rows || (size_t)need > kSmallScratchBytes) {
    std::snprintf(g_err, sizeof g_err,
                  "pca_run_small_static: M = %lld rows of %d (padded) columns need %lld bytes of scratch; the static scratch "
                  "holds %zu bytes, i.e. at most %lld rows at N = %lld", (long long)M, ldr, need, kSmallScratchBytes, max_rows,
                  (long long)N);
    return PCA_EUNSUPPORTED;
  }
  int RPT = 0;
  for (int r : {2, 4, 7})
    if ((long long)NG * r >= M) { RPT = r; break; }
  pca::one_kernel_t fn = pca::one_kernel_lookup(GT, RPT);
  if (!fn) {
    std::snprintf(g_err, sizeof g_err, "pca_run_small_static: no kernel variant for GT = %d, RPT = %d in this build", GT, RPT);
    return PCA_EUNSUPPORTED;
  }
  pca::OneParams p{};
  p.M = (int)M; p.N = (int)N; p.K = K; p.eps = eps; p.max_iter = max_iter; p.algo = algo;
  p.test_mode = 0; p.stag2 = 1; p.out_svd = 0;                       // the library's defaults (PCA_OPT_TEST_MODE / _STAGNATION / _OUTPUT)
  p.ldr = ldr; p.Kpad = (int)round_up(K, 4);
  const bool gs = algo == PCA_ALGO_GS;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = (size_t)round_up((long long)(off + bytes), 16); return (int)o; };
  const size_t rows = (size_t)NG * RPT, KV = (size_t)(p.Kpad | 1);
  p.off_p = take((size_t)ldr * 4);
  p.off_ttil = take(rows * 4);
  p.off_d = take(rows * 4);
  p.off_qs = take((size_t)NG * ldr * 4);
  p.off_red = take((size_t)pca::kThreads * 4);
  p.off_sgrp = take((size_t)NG * 8);
  p.off_q = take((size_t)ldr * 8);
  p.off_B = take((size_t)(2 + p.Kpad) * 8);
  p.off_A = take((size_t)(2 + p.Kpad) * 8);
  p.off_scr = take((size_t)pca::kThreads * 8);
  p.off_vb = take(gs ? rows * KV * 4 : 0);
  p.off_pp = take(gs ? (size_t)ldr * KV * 4 : 0);
  p.off_wp = take(gs ? (size_t)ldr * KV * 4 : 0);
  const size_t smem = off;

  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_cuda(e, "cudaGetDevice");
  if (dev < 0 || dev >= kMaxDevices) {
    std::snprintf(g_err, sizeof g_err, "pca_run_small_static: device ordinal %d outside [0, %d)", dev, kMaxDevices);
    return PCA_EUNSUPPORTED;
  }
  SmallDevice* d = nullptr;
  const int rc = small_setup(dev, &d);
  if (rc != PCA_OK) return rc;
  if (smem > (size_t)d->smem_optin) {
    std::snprintf(g_err, sizeof g_err, "pca_run_small_static: the plan needs %zu bytes of shared memory, the device offers %d", smem,
                  d->smem_optin);
    return PCA_EUNSUPPORTED;
  }
  p.Rrm = static_cast<float*>(d->scratch);                           // the DEVICE address, never the symbol's host-side name
  p.T = T; p.P = P; p.lambda = lambda; p.iters = iters;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const dim3 tgrid((unsigned)ceil_div(M, 32), (unsigned)ceil_div(ldr, 32));
  pca::pca_transpose_in_kernel<<<tgrid, 256, 0, st>>>(X, p.Rrm, M, p.N, ldr);     // R <- X: every word the solve reads
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda(e, "launch of pca_transpose_in_kernel");
  fn<<<1, pca::kThreads, smem, st>>>(p);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda(e, "launch of pca_one_kernel");
  if (R) {
    const dim3 ogrid((unsigned)ceil_div(M, 32), (unsigned)ceil_div(N, 32));
    pca::pca_transpose_plain_kernel<<<ogrid, 256, 0, st>>>(p.Rrm, R, M, p.N, ldr);   // the residual of eq. (4), column-major
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "launch of pca_transpose_plain_kernel");
  }
  return PCA_OK;
}

}  // extern "C"
