// =====================================================================================
// pca_shard.cuh -- row-sharded multi-GPU form of the inner loop.
//
// The path shards by ROWS of R (M >= N): rank g holds R_g (M_g x N), its rows of T / V, and a replica of the
// loading panels P, W.  One inner pass in the single-sweep form of pca_fused.cuh:
//     local   t~_g = R_g p (S5);  q_g = R_g^T t~_g (S2 of the next pass);  s_g = |t~_g|^2;  B_g = V_g^T t~_g (S6)
//     ONE all-reduce of  [ q (N) | s | B (k) ]  = N + k + 1 numbers (fp64)                        <- the only exchange
//     replicated on every rank, from identical reduced numbers: lambda'^2 = s - |B|^2 (S7), test (S8),
//             p~ = q - W B, A = P^T p~, p^ = p~ - P A (S3), p = p^/|p^| (S4)
// and per component: the loads sweep (pending deflation S9 fused with q = R^T t0, S1/S2) and the finalisation
// (t = t~ - V B, v = t/lambda', W_k).  The all-reduce is the CALLER's (torch.distributed: NCCL between GPUs, gloo in the CPU
// tests): every kernel here is rank-local, enqueued step by step by the host API in pca_shard.cu; a step launched after the
// component has converged is a no-op (device-side `done` flag), so the host may look at the flag every few passes only.
// This is the plain NCCL form; the fused form (the LL exchange words of pca_fused.cuh in peer-mapped memory) needs a
// multi-GPU box to be validated and is not built.
// =====================================================================================
#pragma once
#include "pca_fused.cuh"

namespace pca {

struct ShardState {            // device-resident control block of one rank (identical on every rank after each all-reduce)
  double lam, lam2, lam_new;   // lambda' of the previous pass, of the one before, of this one
  double inv_pn;               // 1/|p^| of the loads in flight
  int it;                      // inner passes of the current component
  int done;                    // 1: the current component has converged (or is degenerate): further steps are no-ops
  int degenerate;
  int first;                   // the next reduce belongs to the loads sweep
};

struct ShardParams {
  float* Rrm;        // [Ml][ldr] row-major residual rows of this rank
  float* Vrm;        // [Ml][Kpad] unit score rows (row-major)
  float* T;          // Ml x K column-major (ld = Ml): the caller's output
  float* ttil;       // [Ml] t0 / t~ rows
  float* d;          // [Ml] pending deflation vector rows
  float* p;          // [ldr] unit loads p of the pass in flight
  float* pdef;       // [ldr] loads of the previous component (pending deflation)
  float* Pn;         // [N][Kpad] replicated loadings panel (row-major)
  float* Wn;         // [N][Kpad] replicated W = R^T V panel
  double* praw;      // [N] raw loads q - W B of the pass in flight (for W_k)
  double* part;      // [G][L] per-CTA partials of one sweep
  double* xsend;     // [L] this rank's sums of one sweep: the caller copies them to xbuf and all-reduces xbuf in place
  double* xbuf;      // [L] the reduced numbers (a no-op step leaves xsend as it was, so repeating copy + all-reduce is harmless)
  float* Pout;       // N x K column-major: the caller's P (every rank writes the same values)
  float* lambda;     // K
  int* iters;        // K
  ShardState* st;
  long long Ml;
  int N, K, ldr, GT, G, Mb, Kpad, L;
  double eps;
  int max_iter, algo, test_mode, stag2;
};

// dynamic shared memory of the sweep kernels: p_s[ldr] | ttil_s[Mbp] | d_s[Mbp] | pdef_s[ldr] | qs[NG][ldr] | red_s | sgrp
struct ShardSmem { int off_p, off_ttil, off_d, off_pdef, off_qs, off_red, off_sgrp; size_t bytes; };

// One sweep over this rank's rows.  LOADS: pending deflation + t0 = column k + q = R^T t0 (S9, S1, S2); else t~ = R p (S5),
// q = R^T t~, s, B-partials (S6).  CTA b writes its partials to part[b][0..L): q (N) | s | - | B (k).
template <int NV, bool LOADS>
__global__ void __launch_bounds__(kThreads, 1) pca_shard_sweep_kernel(const ShardParams prm, const ShardSmem sm, int k) {
  if (prm.st->done) return;
  extern __shared__ __align__(16) unsigned char smem[];
  float* p_s = reinterpret_cast<float*>(smem + sm.off_p);
  float* ttil_s = reinterpret_cast<float*>(smem + sm.off_ttil);
  float* d_s = reinterpret_cast<float*>(smem + sm.off_d);
  float* pdef_s = reinterpret_cast<float*>(smem + sm.off_pdef);
  float* qs = reinterpret_cast<float*>(smem + sm.off_qs);
  float* red_s = reinterpret_cast<float*>(smem + sm.off_red);
  double* sgrp = reinterpret_cast<double*>(smem + sm.off_sgrp);
  const int tid = threadIdx.x, b = blockIdx.x, ldr = prm.ldr, N = prm.N, NG = kThreads / prm.GT;
  const long long m0 = (long long)b * prm.Mb;
  const int mb = (int)max(0LL, min((long long)prm.Mb, prm.Ml - m0));
  float* Rb = prm.Rrm + (size_t)m0 * ldr;
  FusedParams fp{};
  fp.GT = prm.GT; fp.ldr = ldr;
  double* out = prm.part + (size_t)b * prm.L;
  const bool gsk = prm.algo == 1 && k > 0;
  double s = 0.0;
  if constexpr (LOADS) {
    for (int n = tid; n < ldr; n += kThreads) pdef_s[n] = prm.pdef[n];
    for (int i = tid; i < mb; i += kThreads) d_s[i] = prm.d[m0 + i];
    __syncthreads();
    for (int i = tid; i < mb; i += kThreads) ttil_s[i] = fmaf(-d_s[i], pdef_s[k], ld_cg(Rb + (size_t)i * ldr + k));   // S1 (C6)
    __syncthreads();
    if (k == 0) sweep_loads<NV, SRC_GLOBAL, DST_NONE, false, true>(fp, Rb, nullptr, mb, ttil_s, d_s, pdef_s, qs);
    else        sweep_loads<NV, SRC_GLOBAL, DST_GLOBAL, true, true>(fp, Rb, nullptr, mb, ttil_s, d_s, pdef_s, qs);
    for (int i = tid; i < mb; i += kThreads) { const double v = (double)ttil_s[i]; s += v * v; }
    s = block_sum(s, reinterpret_cast<double*>(red_s));
  } else {
    const float inv = (float)prm.st->inv_pn;
    for (int n = tid; n < ldr; n += kThreads) p_s[n] = prm.p[n] * inv;
    __syncthreads();
    sweep_fused<NV, SRC_GLOBAL>(fp, Rb, nullptr, mb, p_s, ttil_s, qs, red_s, sgrp, false);
    for (int g = 0; g < NG; ++g) s += sgrp[g];
  }
  for (int i = tid; i < mb; i += kThreads) prm.ttil[m0 + i] = ttil_s[i];
  for (int n = tid; n < N; n += kThreads) {
    double a = 0.0;
    for (int g = 0; g < NG; ++g) a += (double)qs[(size_t)g * ldr + n];
    out[n] = a;
  }
  if (tid == 0) { out[N] = s; out[N + 1] = 0.0; }
  // B-partials (S6): 32 consecutive columns j per warp (coalesced rows of the row-major V), the 16 warps split the rows
  __syncthreads();                                           // qs is consumed: reuse it as [kWarps][32] floats
  float* bred = qs;
  for (int jb = 0; jb < prm.Kpad; jb += 32) {
    const int lane = tid & 31, w = tid >> 5, j = jb + lane;
    float af = 0.f;
    if (!LOADS && gsk && j < k) {
      const float* vr = prm.Vrm + (size_t)m0 * prm.Kpad + j;
      for (int i = w; i < mb; i += kWarps) af = fmaf(vr[(size_t)i * prm.Kpad], ttil_s[i], af);
    }
    bred[w * 32 + lane] = af;
    __syncthreads();
    if (w == 0 && j < prm.Kpad) {
      double a = 0.0;
      for (int q2 = 0; q2 < kWarps; ++q2) a += (double)bred[q2 * 32 + lane];   // fixed order
      out[N + 2 + j] = a;
    }
    __syncthreads();
  }
}

// xbuf[j] = sum over the CTAs of part[b][j], fixed order
// (32 columns per CTA, 8 groups of parts per column: coalesced 256-byte rows, 8 independent chains)
static __global__ void __launch_bounds__(256) pca_shard_reduce_kernel(const ShardParams prm) {
  if (prm.st->done) return;
  __shared__ double red[8][33];
  const int jl = threadIdx.x & 31, pg = threadIdx.x >> 5;
  const int j = blockIdx.x * 32 + jl;
  double a = 0.0;
  if (j < prm.L)
    for (int b = pg; b < prm.G; b += 8) a += prm.part[(size_t)b * prm.L + j];
  red[pg][jl] = a;
  __syncthreads();
  if (pg == 0 && j < prm.L) {
    double t = 0.0;
    for (int q = 0; q < 8; ++q) t += red[q][jl];
    prm.xsend[j] = t;
  }
}

// The replicated loads side (one CTA): consumes the all-reduced [ q | s | B ].
static __global__ void __launch_bounds__(1024, 1) pca_shard_nside_kernel(const ShardParams prm, int k) {
  ShardState* st = prm.st;
  if (st->done) return;
  __shared__ double scr[40];
  __shared__ double ctl[4];
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, w = tid >> 5;
  const int N = prm.N, Kpad = prm.Kpad;
  const bool gsk = prm.algo == 1 && k > 0;
  const double* q = prm.xbuf;
  const double* B = prm.xbuf + N + 2;
  const bool first = st->first != 0;
  auto bsum = [&](double v) -> double {                      // block sum, fixed order
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) scr[w] = v;
    __syncthreads();
    if (w == 0) {
      double x = (lane < (nthr >> 5)) ? scr[lane] : 0.0;
      x = warp_sum(x);
      if (lane == 0) scr[32] = x;
    }
    __syncthreads();
    return scr[32];
  };
  // S7 / S8
  double bb = 0.0;
  if (gsk && !first)
    for (int j = tid; j < k; j += nthr) bb += B[j] * B[j];
  bb = bsum(bb);
  if (tid == 0) {
    const double s = q[N];
    int stt = 0;
    double ln = 0.0;
    if (first) {
      if (!(s > 0.0)) stt = 2;                                // zero start column (C7)
    } else {
      const double l2 = s - bb;                               // |t~ - V B|^2, V orthonormal
      if (!(l2 > 0.0)) stt = 2;
      else {
        ln = sqrt(l2);                                        // S7
        if (pca_stagnated(st->lam, st->lam2, ln, prm.eps, prm.test_mode, prm.stag2) || st->it >= prm.max_iter) stt = 1;   // S8
      }
    }
    ctl[0] = ln; ctl[1] = (double)stt;
  }
  __syncthreads();
  const int stt = (int)ctl[1];
  const double ln = ctl[0];
  // p~ = q - W B (linearity, see pca_fused.cuh), kept in fp64 for W_k
  for (int n = tid; n < N; n += nthr) {
    double v = q[n];
    if (gsk && !first) {
      const float* wr = prm.Wn + (size_t)n * Kpad;
      double c = 0.0;
      for (int j = 0; j < k; ++j) c += (double)wr[j] * B[j];
      v -= c;
    }
    prm.praw[n] = v;
  }
  __syncthreads();
  if (stt == 2) {
    if (tid == 0) { st->done = 1; st->degenerate = 1; }
    return;
  }
  if (stt == 1) {
    if (tid == 0) { st->lam_new = ln; st->done = 1; }
    return;
  }
  // S3: A = P^T p~ ; p^ = p~ - P A.  A in shared memory (k <= 1024 per chunk of the block)
  __shared__ double A_s[1024];
  __shared__ double red32[32][33];
  if (gsk) {
    for (int j0 = 0; j0 < k; j0 += 1024) {
      // A[j] = sum_n P[n,j] p~[n]: 32 consecutive j per warp-row (coalesced rows of the row-major panel), the 32 warps split n
      for (int jb = j0; jb < min(k, j0 + 1024); jb += 32) {
        const int j = jb + lane;
        double a = 0.0;
        if (j < k)
          for (int n = w; n < N; n += (nthr >> 5)) a += (double)prm.Pn[(size_t)n * Kpad + j] * prm.praw[n];
        __syncthreads();                                    // red32 free
        red32[w][lane] = a;
        __syncthreads();
        if (w == 0 && j < k) {
          double t = 0.0;
          for (int q2 = 0; q2 < (nthr >> 5); ++q2) t += red32[q2][lane];   // fixed order
          A_s[j - j0] = t;
        }
      }
      __syncthreads();
      for (int n = tid; n < N; n += nthr) {
        const float* pr = prm.Pn + (size_t)n * Kpad;
        double c = 0.0;
        for (int j = j0; j < min(k, j0 + 1024); ++j) c += (double)pr[j] * A_s[j - j0];
        prm.xbuf[n] = prm.praw[n] - c;                        // p^ (the reduced q is consumed; praw keeps p~ for W_k)
      }
      __syncthreads();
      if (j0 + 1024 < k)
        for (int n = tid; n < N; n += nthr) prm.praw[n] = prm.xbuf[n];   // (K > 1024: project chunk by chunk)
      __syncthreads();
    }
  } else {
    for (int n = tid; n < N; n += nthr) prm.xbuf[n] = prm.praw[n];
  }
  __syncthreads();
  double q2 = 0.0;
  for (int n = tid; n < N; n += nthr) { const float v = (float)prm.xbuf[n]; prm.p[n] = v; q2 += (double)v * (double)v; }
  for (int n = N + tid; n < prm.ldr; n += nthr) prm.p[n] = 0.f;
  q2 = bsum(q2);
  if (tid == 0) {
    if (!(q2 > 0.0)) { st->done = 1; st->degenerate = 1; }
    else {
      st->inv_pn = 1.0 / sqrt(q2);
      if (!first) { st->lam2 = st->lam; st->lam = ln; }
      st->first = 0;
      st->it += 1;                                            // the sweep that follows is pass number `it`
    }
  }
}

// Component k is done on every rank: rows of t, v, T, the replicated P / W columns, lambda, iters; state reset.
static __global__ void __launch_bounds__(256) pca_shard_finalize_kernel(const ShardParams prm, int k, int nrowblocks) {
  const ShardState* st = prm.st;
  const int tid = threadIdx.x, Kpad = prm.Kpad, N = prm.N;
  const bool gs = prm.algo == 1, gsk = gs && k > 0;
  const double* B = prm.xbuf + N + 2;
  const double lam = st->lam_new;
  if ((int)blockIdx.x < nrowblocks) {
    const long long r = (long long)blockIdx.x * blockDim.x + tid;
    if (r >= prm.Ml) return;
    if (st->degenerate) {
      prm.T[(size_t)k * prm.Ml + r] = 0.f; prm.d[r] = 0.f;
      if (gs) prm.Vrm[(size_t)r * Kpad + k] = 0.f;
      return;
    }
    float t = prm.ttil[r];
    if (gsk) {                                                // t = t~ - V_(k) B
      float corr = 0.f;
      const float* vr = prm.Vrm + (size_t)r * Kpad;
      for (int j = 0; j < k; ++j) corr = fmaf(vr[j], (float)B[j], corr);
      t -= corr;
    }
    const float inv = (float)(1.0 / lam);
    prm.d[r] = t;                                             // S9: R -= lambda v p^T  /  R -= t p^T
    prm.T[(size_t)k * prm.Ml + r] = gs ? t * inv : t;         // GS-PCA: unit v until the epilogue S10
    if (gs) prm.Vrm[(size_t)r * Kpad + k] = t * inv;
  } else {                                                    // the replicated loads side (same values on every rank)
    const int n = ((int)blockIdx.x - nrowblocks) * blockDim.x + tid;
    if (n < prm.ldr) {
      const float pk = (st->degenerate || n >= N) ? 0.f : prm.p[n] * (float)st->inv_pn;
      prm.pdef[n] = pk;
      if (n < N) {
        prm.Pout[(size_t)k * N + n] = pk;
        prm.Pn[(size_t)n * Kpad + k] = pk;
        prm.Wn[(size_t)n * Kpad + k] = (st->degenerate || !gs) ? 0.f : (float)(prm.praw[n] / lam - lam * (double)pk);   // W_k = R_(k+1)^T v_k
      }
    }
    if (n == 0) {
      prm.lambda[k] = st->degenerate ? 0.f : (float)lam;
      prm.iters[k] = st->degenerate ? 0 : st->it;
    }
  }
}

// state for the next component (after the finalize kernel)
static __global__ void pca_shard_reset_kernel(ShardState* st) {
  st->lam = 0.0; st->lam2 = 0.0; st->lam_new = 0.0; st->inv_pn = 0.0; st->it = 0; st->done = 0; st->degenerate = 0; st->first = 1;
}

// S10 epilogue (GS-PCA): T <- V Lambda on this rank's rows; and the residual rows of eq. (4) with the last deflation applied
static __global__ void __launch_bounds__(256) pca_shard_epilogue_kernel(const ShardParams prm, float* Rout /*Ml x N col-major or null*/) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= prm.Ml) return;
  const float dr = prm.d[r];
  if (Rout) {
    const float* row = prm.Rrm + (size_t)r * prm.ldr;
    for (int n = 0; n < prm.N; ++n) Rout[(size_t)n * prm.Ml + r] = fmaf(-dr, prm.pdef[n], row[n]);
  }
  if (prm.algo == 1)
    for (int kk = 0; kk < prm.K; ++kk) prm.T[(size_t)kk * prm.Ml + r] *= prm.lambda[kk];
}

// column sums of this rank's rows (centring S0 across ranks: the caller all-reduces the N sums) and the subtraction
static __global__ void __launch_bounds__(256) pca_shard_colsum_kernel(const float* __restrict__ X, long long Ml, int N, double* __restrict__ sums) {
  __shared__ double red[8];
  const int n = blockIdx.x, tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  double s = 0.0;
  for (long long i = tid; i < Ml; i += 256) s += (double)__ldcg(X + (size_t)n * Ml + i);
  s = warp_sum(s);
  if (lane == 0) red[w] = s;
  __syncthreads();
  if (tid == 0) { double t = 0.0; for (int i = 0; i < 8; ++i) t += red[i]; sums[n] = t; }
}
static __global__ void __launch_bounds__(256) pca_shard_center_apply_kernel(float* __restrict__ X, long long Ml, int N, const double* __restrict__ sums,
                                                                            double inv_M_total) {
  const int n = blockIdx.y;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < Ml) X[(size_t)n * Ml + i] = (float)((double)X[(size_t)n * Ml + i] - sums[n] * inv_M_total);
}

}  // namespace pca
