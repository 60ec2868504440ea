// =====================================================================================
// pca_shard.cu -- host side of the row-sharded multi-GPU entry points declared in include/pca.h (pca_shard_*):
// rank-local plan, workspace layout and step-by-step launches of the kernels in pca_shard.cuh.  The all-reduce between
// the steps is the caller's (torch.distributed).  No torch types, nothing prints, throws or exits.
// =====================================================================================
#include "../../include/pca.h"

#include <cuda_runtime.h>

#include <cstdint>
#include <new>

#include "pca_shard.cuh"

using pca::ShardParams;
using pca::ShardSmem;
using pca::ShardState;

namespace {
inline long long round_up(long long v, long long a) { return (v + a - 1) / a * a; }
inline long long ceil_div(long long a, long long b) { return (a + b - 1) / b; }
typedef void (*sweep_fn)(const ShardParams, const ShardSmem, int);
struct SweepVariant { int nv; sweep_fn loads, fused; };
#define PCA_SV(NV) {NV, pca::pca_shard_sweep_kernel<NV, true>, pca::pca_shard_sweep_kernel<NV, false>}
const SweepVariant kSweeps[] = {PCA_SV(1), PCA_SV(2), PCA_SV(3), PCA_SV(4)};
#undef PCA_SV
}  // namespace

struct pca_shard {
  ShardParams p{};
  ShardSmem sm{};
  const SweepVariant* var = nullptr;
  size_t ws_bytes = 0;
  size_t off_rrm = 0, off_vrm = 0, off_ttil = 0, off_d = 0, off_p = 0, off_pdef = 0, off_pn = 0, off_wn = 0, off_praw = 0,
         off_part = 0, off_xsend = 0, off_xbuf = 0, off_st = 0;
  void* ws = nullptr;
  bool begun = false;
  bool attr_set[2] = {false, false};
  int smem_optin = 0;
  int last_cuda = 0;
};

#define SH_CUDA(c, expr)                                                  \
  do {                                                                    \
    cudaError_t e__ = (expr);                                             \
    if (e__ != cudaSuccess) { (c)->last_cuda = (int)e__; return PCA_ECUDA; } \
  } while (0)

extern "C" {

int pca_shard_create(pca_shard** out, int64_t M_local, int64_t N, int K, double eps, int max_iter, int algo) {
  if (!out) return PCA_EINVAL;
  *out = nullptr;
  if (M_local < 1 || N < 1 || K < 1 || (int64_t)K > N || !(eps >= 0.0) || max_iter < 1) return PCA_EINVAL;
  if (algo != PCA_ALGO_NIPALS && algo != PCA_ALGO_GS) return PCA_EINVAL;
  if (K > 1024 || N > 16 * pca::kThreads) return PCA_EUNSUPPORTED;   // loads-side projection in one chunk; NV <= 4
  int dev = 0, sms = 0, smem_optin = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
    return PCA_ECUDA;                                               // no CUDA device: there is no CPU fallback
  pca_shard* c = new (std::nothrow) pca_shard();
  if (!c) return PCA_EINVAL;
  c->smem_optin = smem_optin;
  ShardParams& p = c->p;
  p.Ml = M_local; p.N = (int)N; p.K = K; p.eps = eps; p.max_iter = max_iter; p.algo = algo; p.test_mode = 0; p.stag2 = 1;
  int GT = 32;
  while ((long long)16 * GT < N) GT *= 2;
  const int NV = (int)ceil_div(N, 4LL * GT);
  p.GT = GT; p.ldr = 4 * GT * NV;
  p.Kpad = (int)round_up(K, 4);
  p.L = (int)round_up(N + 2 + p.Kpad, 2);
  for (const SweepVariant& v : kSweeps)
    if (v.nv == NV) c->var = &v;
  if (!c->var) { delete c; return PCA_EUNSUPPORTED; }
  // CTAs: as many as SMs, fewer if the rows of a CTA (t~, d in shared memory) would not fit otherwise
  int G = (int)(M_local < sms ? M_local : sms);
  for (;;) {
    p.G = G; p.Mb = (int)ceil_div(M_local, G);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = (size_t)round_up((long long)(off + bytes), 16); return (int)o; };
    const size_t mbp = (size_t)round_up(p.Mb, 4);
    c->sm.off_p = take((size_t)p.ldr * 4);
    c->sm.off_ttil = take(mbp * 4);
    c->sm.off_d = take(mbp * 4);
    c->sm.off_pdef = take((size_t)p.ldr * 4);
    c->sm.off_qs = take((size_t)(pca::kThreads / GT) * p.ldr * 4);
    c->sm.off_red = take((size_t)2 * pca::kWarps * pca::kRB * 4 + 160);
    c->sm.off_sgrp = take((size_t)(pca::kThreads / GT) * 8);
    c->sm.bytes = off;
    if (off <= (size_t)smem_optin) break;
    delete c;
    return PCA_EUNSUPPORTED;                                        // (a rank's row block per CTA must fit: M_local/148 rows)
  }
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = (size_t)round_up((long long)(off + bytes), 256); return o; };
  c->off_rrm = take((size_t)M_local * p.ldr * 4);
  c->off_vrm = take(algo == PCA_ALGO_GS ? (size_t)M_local * p.Kpad * 4 : 0);
  c->off_ttil = take((size_t)M_local * 4);
  c->off_d = take((size_t)M_local * 4);
  c->off_p = take((size_t)p.ldr * 4);
  c->off_pdef = take((size_t)p.ldr * 4);
  c->off_pn = take((size_t)N * p.Kpad * 4);
  c->off_wn = take((size_t)N * p.Kpad * 4);
  c->off_praw = take((size_t)N * 8);
  c->off_part = take((size_t)p.G * p.L * 8);
  c->off_xsend = take((size_t)p.L * 8);
  c->off_xbuf = take((size_t)p.L * 8);
  c->off_st = take(sizeof(ShardState));
  c->ws_bytes = off;
  *out = c;
  return PCA_OK;
}

size_t pca_shard_workspace_bytes(const pca_shard* c) { return c ? c->ws_bytes : 0; }

int pca_shard_set_workspace(pca_shard* c, void* dev, size_t bytes) {
  if (!c || !dev) return PCA_EINVAL;
  if ((reinterpret_cast<uintptr_t>(dev) & 255u) != 0) return PCA_EALIGN;
  if (bytes < c->ws_bytes) return PCA_EWORKSPACE;
  unsigned char* ws = static_cast<unsigned char*>(dev);
  c->ws = dev;
  ShardParams& p = c->p;
  p.Rrm = reinterpret_cast<float*>(ws + c->off_rrm);
  p.Vrm = reinterpret_cast<float*>(ws + c->off_vrm);
  p.ttil = reinterpret_cast<float*>(ws + c->off_ttil);
  p.d = reinterpret_cast<float*>(ws + c->off_d);
  p.p = reinterpret_cast<float*>(ws + c->off_p);
  p.pdef = reinterpret_cast<float*>(ws + c->off_pdef);
  p.Pn = reinterpret_cast<float*>(ws + c->off_pn);
  p.Wn = reinterpret_cast<float*>(ws + c->off_wn);
  p.praw = reinterpret_cast<double*>(ws + c->off_praw);
  p.part = reinterpret_cast<double*>(ws + c->off_part);
  p.xsend = reinterpret_cast<double*>(ws + c->off_xsend);
  p.xbuf = reinterpret_cast<double*>(ws + c->off_xbuf);
  p.st = reinterpret_cast<ShardState*>(ws + c->off_st);
  c->begun = false;
  return PCA_OK;
}

int pca_shard_exchange(const pca_shard* c, double** send, double** recv, int64_t* count) {
  if (!c || !send || !recv || !count) return PCA_EINVAL;
  if (!c->ws) return PCA_EWORKSPACE;
  *send = c->p.xsend; *recv = c->p.xbuf; *count = c->p.L;
  return PCA_OK;
}

int pca_shard_colsums(pca_shard* c, const float* X_local, double* sums, void* stream) {
  if (!c || !X_local || !sums) return PCA_EINVAL;
  pca::pca_shard_colsum_kernel<<<(unsigned)c->p.N, 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(X_local, c->p.Ml, c->p.N, sums);
  SH_CUDA(c, cudaGetLastError());
  return PCA_OK;
}

int pca_shard_center(pca_shard* c, float* X_local, const double* sums_reduced, int64_t M_total, void* stream) {
  if (!c || !X_local || !sums_reduced || M_total < c->p.Ml) return PCA_EINVAL;
  const dim3 grid((unsigned)ceil_div(c->p.Ml, 256), (unsigned)c->p.N);
  pca::pca_shard_center_apply_kernel<<<grid, 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(X_local, c->p.Ml, c->p.N, sums_reduced,
                                                                                              1.0 / (double)M_total);
  SH_CUDA(c, cudaGetLastError());
  return PCA_OK;
}

int pca_shard_begin(pca_shard* c, const float* X_local, float* T, float* P, float* lambda, int32_t* iters, void* stream) {
  if (!c || !X_local || !T || !P || !lambda || !iters) return PCA_EINVAL;
  if (!c->ws) return PCA_EWORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  ShardParams& p = c->p;
  p.T = T; p.Pout = P; p.lambda = lambda; p.iters = iters;
  unsigned char* ws = static_cast<unsigned char*>(c->ws);
  SH_CUDA(c, cudaMemsetAsync(ws + c->off_vrm, 0, c->ws_bytes - c->off_vrm, st));      // everything but R: d, pdef, panels, state
  const dim3 tgrid((unsigned)ceil_div(p.Ml, 32), (unsigned)ceil_div(p.ldr, 32));
  pca::pca_transpose_in_kernel<<<tgrid, 256, 0, st>>>(X_local, p.Rrm, p.Ml, p.N, p.ldr);   // R <- X
  SH_CUDA(c, cudaGetLastError());
  pca::pca_shard_reset_kernel<<<1, 1, 0, st>>>(p.st);
  SH_CUDA(c, cudaGetLastError());
  c->begun = true;
  return PCA_OK;
}

static int launch_sweep(pca_shard* c, bool loads, int k, cudaStream_t st) {
  const ShardParams& p = c->p;
  sweep_fn fn = loads ? c->var->loads : c->var->fused;
  if (!c->attr_set[loads ? 0 : 1]) {                                  // once per context and kernel (the call is not cheap)
    // (the attribute belongs to the FUNCTION, not to this context: ask for the device maximum, so that contexts with different
    //  shared-memory needs -- the shards of one process -- do not lower it for each other)
    SH_CUDA(c, cudaFuncSetAttribute(reinterpret_cast<const void*>(fn), cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin));
    c->attr_set[loads ? 0 : 1] = true;
  }
  fn<<<(unsigned)p.G, pca::kThreads, c->sm.bytes, st>>>(p, c->sm, k);
  SH_CUDA(c, cudaGetLastError());
  pca::pca_shard_reduce_kernel<<<(unsigned)ceil_div(p.L, 32), 256, 0, st>>>(p);
  SH_CUDA(c, cudaGetLastError());
  return PCA_OK;
}

int pca_shard_component(pca_shard* c, int k, void* stream) {
  if (!c || k < 0 || k >= c->p.K) return PCA_EINVAL;
  if (!c->begun) return PCA_EWORKSPACE;
  return launch_sweep(c, true, k, reinterpret_cast<cudaStream_t>(stream));
}

int pca_shard_pass(pca_shard* c, int k, void* stream) {
  if (!c || k < 0 || k >= c->p.K) return PCA_EINVAL;
  if (!c->begun) return PCA_EWORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  pca::pca_shard_nside_kernel<<<1, 1024, 0, st>>>(c->p, k);
  SH_CUDA(c, cudaGetLastError());
  return launch_sweep(c, false, k, st);
}

int pca_shard_done(pca_shard* c, int32_t* done_host, void* stream) {
  if (!c || !done_host) return PCA_EINVAL;
  if (!c->begun) return PCA_EWORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  int flag = 0;
  SH_CUDA(c, cudaMemcpyAsync(&flag, &c->p.st->done, sizeof(int), cudaMemcpyDeviceToHost, st));
  SH_CUDA(c, cudaStreamSynchronize(st));
  *done_host = flag;
  return PCA_OK;
}

int pca_shard_finish_component(pca_shard* c, int k, void* stream) {
  if (!c || k < 0 || k >= c->p.K) return PCA_EINVAL;
  if (!c->begun) return PCA_EWORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const int nrow = (int)ceil_div(c->p.Ml, 256), ncol = (int)ceil_div(c->p.ldr, 256);
  pca::pca_shard_finalize_kernel<<<(unsigned)(nrow + ncol), 256, 0, st>>>(c->p, k, nrow);
  SH_CUDA(c, cudaGetLastError());
  pca::pca_shard_reset_kernel<<<1, 1, 0, st>>>(c->p.st);
  SH_CUDA(c, cudaGetLastError());
  return PCA_OK;
}

int pca_shard_end(pca_shard* c, float* R_local, void* stream) {
  if (!c) return PCA_EINVAL;
  if (!c->begun) return PCA_EWORKSPACE;
  pca::pca_shard_epilogue_kernel<<<(unsigned)ceil_div(c->p.Ml, 256), 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(c->p, R_local);
  SH_CUDA(c, cudaGetLastError());
  return PCA_OK;
}

void pca_shard_destroy(pca_shard* c) { delete c; }

int pca_shard_last_cuda_error(const pca_shard* c) { return c ? c->last_cuda : 0; }

}  // extern "C"
