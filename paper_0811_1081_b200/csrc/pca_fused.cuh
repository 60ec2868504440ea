// =====================================================================================
// pca_fused.cuh -- single-sweep persistent solve kernel.
//
// One inner pass of NIPALS-PCA / GS-PCA needs t = R p and then p' = R^T t (PAPER.md:564,:562 /
// :1028,:1023).  A CTA that owns a ROW BLOCK of R (all N columns of its rows) can form its rows
// of t locally and, with the rows still in registers, its partial of R^T t: R is read ONCE per
// inner pass instead of twice, and there is one exchange of partials per pass instead of two.
// The iterates are the paper's (same statement order, same start vector, same test); only the
// loop is rotated: the sweep that produces lambda' also produces the raw loads of the next pass.
//
// Layout: the residual is kept ROW-major in the workspace (Rrm[m][ldr], ldr >= N padded with
// zeros) so that a row is one contiguous, 128-bit-coalesced stream and a thread can own fixed
// columns.  X (column-major, the ABI layout) is transposed in once and the residual of eq. (4)
// is transposed out once (pca_transpose_in/out kernels below); both are outside the inner loop.
//
// GS-PCA's scores-side projection t = t~ - V B sits between the two
// products; by linearity  R^T (t~ - V B) = R^T t~ - W B  with  W = R^T V_(k)  (N x k).  W's column j
// is created when component j finishes, from quantities the sweep has already produced:
//   W_j = R_(j+1)^T v_j = (R_j^T t_j) / lambda_j - lambda_j p_j        (deflation R_(j+1) = R_j - lambda_j v_j p_j^T)
// and is not touched afterwards (later deflations change it by lambda_i p_i (v_i^T v_j), and
// v_i^T v_j is the rounding-level orthogonality defect of the scores).  The loads-side projection
// p^ = p~ - P A, A = P_(k)^T p~ is taken on the actual vector, as in the paper.
// lambda'^2 = ||t~ - V B||^2 = ||t~||^2 - ||B||^2 (V orthonormal), so lambda', B and the raw loads all
// come out of ONE exchange; t itself is only formed when the component has converged.
//
// Per component k:
//   t0 <- column k of the deflated residual                                   (S1)
//   LOADS sweep : R <- R - d p_prev^T (pending deflation S9, stored), q = R^T t0, s = |t0|^2
//   loop: [X1] s, B known everywhere -> lambda', test (S7, S8) -> owners: p~ = q - W B, A-partials
//         [X2] A -> p^ = p~ - P A, |p^|^2 partials (S3)     (GS-PCA and k > 0 only)
//         [X3] p = p^/|p^| everywhere (S4) -> FUSED sweep: t~ = R p (S5), q = R^T t~ (S2 of the
//              next pass), s = |t~|^2, B-partials = V^T t~ (S6)
//   finalize: t = t~ - V B, v = t/lambda', store T, P, lambda, iters, W_k; d <- t
// [X1..X3] are grid barriers; every CTA takes the same decisions from the same reduced values.
// =====================================================================================
#pragma once
#include "pca_device.cuh"

namespace pca {

struct FusedParams {
  float* Rrm;            // M x ldr row-major residual (workspace)
  float* T;              // M x K col-major (V until the epilogue for GS-PCA)
  float* P;              // N x K col-major
  float* lambda;         // K
  int* iters;            // K
  long long M;
  int N, K;
  double eps;
  int max_iter;
  int algo;              // 0 NIPALS, 1 GS
  int G;                 // CTAs
  int Mb;                // rows per CTA
  int ldr;               // row stride of Rrm / slab (floats) = 4*GT*NV
  int GT;                // threads that share one row (power of two, 32..512)
  int Ns, Gs;            // columns per slice owner, number of owners
  int Kpad;
  float* Qpart;          // [2][G][ldr]  partial raw loads (double-buffered by sweep parity)
  float* Bpart;          // [2][G][Kpad] partial B
  double* Spart;         // [2][G]       partial |t~|^2
  float* Apart;          // [Gs][Kpad]   partial A
  float* pvec;           // [ldr]        p^ (orthogonalised, not normalised)
  double* Npart;         // [Gs]         partial |p^|^2
  float* W;              // [ldr][Kpad]  W = R^T V
  unsigned long long* bar;
  unsigned long long* trace;  // optional phase trace (PCA_OPT_TRACE): [0] = records written, then records
  int trace_cap;              // capacity in records (0 = off)
  // shared-memory carve-up (byte offsets)
  int off_p, off_pdef, off_ttil, off_d, off_qs, off_red, off_sgrp, off_B, off_A, off_scr, off_praw, off_lam, off_slab;
};

constexpr int kRB = 4;   // rows per batch

// Phase trace (include/pca.h, PCA_OPT_TRACE): thread 0 of CTA 0 appends (phase << 56) | clock64().
enum { TR_COMPONENT = 1, TR_LOADS_DONE = 2, TR_X1 = 3, TR_TEST = 4, TR_QSLICE = 5, TR_APART = 6, TR_X2 = 7,
       TR_PHAT = 8, TR_X3 = 9, TR_PREADY = 10, TR_SWEEP = 11, TR_PUBLISHED = 12, TR_FINAL = 13 };
__device__ __forceinline__ void trace_mark(const FusedParams& prm, int& tn, int phase) {
  if (prm.trace_cap > 0 && blockIdx.x == 0 && threadIdx.x == 0 && tn < prm.trace_cap) {
    prm.trace[1 + tn] = ((unsigned long long)phase << 56) | ((unsigned long long)clock64() & 0x00ffffffffffffffULL);
    ++tn;
  }
}

__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

__device__ __forceinline__ float4 ld_stream4(const float* p) { return __ldcg(reinterpret_cast<const float4*>(p)); }

__device__ __forceinline__ float dot4(const float4 a, const float4 b, float acc) {
  acc = fmaf(a.x, b.x, acc);
  acc = fmaf(a.y, b.y, acc);
  acc = fmaf(a.z, b.z, acc);
  acc = fmaf(a.w, b.w, acc);
  return acc;
}
__device__ __forceinline__ void axpy4(float4& q, const float4 x, const float a) {
  q.x = fmaf(x.x, a, q.x);
  q.y = fmaf(x.y, a, q.y);
  q.z = fmaf(x.z, a, q.z);
  q.w = fmaf(x.w, a, q.w);
}

// ------------------------------------------------------------------------------------ LOADS sweep
// For every owned row r:  x = src[r,:];  (DEFL) x -= d[r]*pdef;  (DST) dst[r,:] = x;  (DOT) q += x*t0[r].
// Leaves the per-group partial q in qs[g][ldr] (DOT) and ends with __syncthreads().
template <int NV, int SRC, int DST, bool DEFL, bool DOT>
__device__ __forceinline__ void sweep_loads(const FusedParams& prm, float* Rb, float* slab, int mb,
                                            const float* t0_s, const float* d_s, const float* pdef_s, float* qs) {
  const int GT = prm.GT, NG = kThreads / GT, ldr = prm.ldr;
  const int tid = threadIdx.x, g = tid / GT, gl = tid - g * GT;
  float4 pd[NV], q[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    pd[v] = DEFL ? *reinterpret_cast<const float4*>(pdef_s + 4 * (gl + GT * v)) : make_float4(0.f, 0.f, 0.f, 0.f);
    q[v] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  const int nb = (mb + kRB - 1) / kRB;
  for (int bi = g; bi < nb; bi += NG) {
    const int r0 = bi * kRB;
    float4 x[kRB][NV];
#pragma unroll
    for (int i = 0; i < kRB; ++i) {
      const int r = r0 + i;
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const int c = 4 * (gl + GT * v);
        if (r < mb) {
          if constexpr (SRC == SRC_GLOBAL) x[i][v] = ld_stream4(Rb + (size_t)r * ldr + c);
          else x[i][v] = *reinterpret_cast<const float4*>(slab + (size_t)r * ldr + c);
        } else {
          x[i][v] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
      }
    }
#pragma unroll
    for (int i = 0; i < kRB; ++i) {
      const int r = r0 + i;
      if (r < mb) {
        const float dr = DEFL ? -d_s[r] : 0.f;
        const float tr = DOT ? t0_s[r] : 0.f;
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const int c = 4 * (gl + GT * v);
          if constexpr (DEFL) axpy4(x[i][v], pd[v], dr);
          if constexpr (DST == DST_GLOBAL) *reinterpret_cast<float4*>(Rb + (size_t)r * ldr + c) = x[i][v];
          if constexpr (DST == DST_SLAB) *reinterpret_cast<float4*>(slab + (size_t)r * ldr + c) = x[i][v];
          if constexpr (DOT) axpy4(q[v], x[i][v], tr);
        }
      }
    }
  }
  if constexpr (DOT) {
#pragma unroll
    for (int v = 0; v < NV; ++v) *reinterpret_cast<float4*>(qs + (size_t)g * ldr + 4 * (gl + GT * v)) = q[v];
  }
  __syncthreads();
}

// ------------------------------------------------------------------------------------ FUSED sweep
// For every owned row r:  t~[r] = sum_n R[r,n] p[n]   (S5);   q[n] += R[r,n] t~[r]   (S2 of the next pass).
// The GT threads of a group share a row; a group takes kRB rows at a time, keeps them in
// registers, reduces the kRB partial dots across the group (shuffle butterfly + one named barrier
// when the group spans several warps) and reuses the registers for the second product.
// Leaves qs[g][ldr], ttil_s[rows], sgrp[g] = sum t~^2 (fp64); ends with __syncthreads().
template <int NV, int SRC>
__device__ __forceinline__ void sweep_fused(const FusedParams& prm, const float* Rb, const float* slab, int mb,
                                            const float* p_s, float* ttil_s, float* qs, float* red_s, double* sgrp,
                                            bool rev) {
  const int GT = prm.GT, NG = kThreads / GT, WG = GT >> 5, ldr = prm.ldr;
  const int tid = threadIdx.x, g = tid / GT, gl = tid - g * GT, lane = tid & 31, wg = gl >> 5;
  float4 pr[NV], q[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    pr[v] = *reinterpret_cast<const float4*>(p_s + 4 * (gl + GT * v));
    q[v] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  double sacc = 0.0;
  const int nb = (mb + kRB - 1) / kRB;
  int parity = 0;
  for (int bq = g; bq < nb; bq += NG) {
    const int bi = rev ? (nb - 1 - bq) : bq;
    const int r0 = bi * kRB;
    float4 x[kRB][NV];
#pragma unroll
    for (int i = 0; i < kRB; ++i) {
      const int r = r0 + i;
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const int c = 4 * (gl + GT * v);
        if (r < mb) {
          if constexpr (SRC == SRC_GLOBAL) x[i][v] = ld_stream4(Rb + (size_t)r * ldr + c);
          else x[i][v] = *reinterpret_cast<const float4*>(slab + (size_t)r * ldr + c);
        } else {
          x[i][v] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
      }
    }
    float part[kRB];
#pragma unroll
    for (int i = 0; i < kRB; ++i) {
      float a = 0.f;
#pragma unroll
      for (int v = 0; v < NV; ++v) a = dot4(x[i][v], pr[v], a);
      part[i] = a;
    }
    // butterfly over the warp: 4 values -> lanes 0,8,16,24 (and their 8-lane groups) hold rows 0..3
    const bool hi = (lane & 16) != 0;
    float k0 = hi ? part[2] : part[0], k1 = hi ? part[3] : part[1];
    const float s0 = hi ? part[0] : part[2], s1 = hi ? part[1] : part[3];
    k0 += __shfl_xor_sync(0xffffffffu, s0, 16);
    k1 += __shfl_xor_sync(0xffffffffu, s1, 16);
    const bool h8 = (lane & 8) != 0;
    float kk = h8 ? k1 : k0;
    const float ss = h8 ? k0 : k1;
    kk += __shfl_xor_sync(0xffffffffu, ss, 8);
    kk += __shfl_xor_sync(0xffffffffu, kk, 4);
    kk += __shfl_xor_sync(0xffffffffu, kk, 2);
    kk += __shfl_xor_sync(0xffffffffu, kk, 1);
    float tt[kRB];
    if (WG == 1) {
#pragma unroll
      for (int i = 0; i < kRB; ++i) tt[i] = __shfl_sync(0xffffffffu, kk, 8 * i);
    } else {
      float* rs = red_s + (size_t)parity * (kWarps * kRB) + (size_t)(g * WG) * kRB;
      if ((lane & 7) == 0) rs[wg * kRB + (lane >> 3)] = kk;
      named_bar_sync(1 + g, GT);
#pragma unroll
      for (int i = 0; i < kRB; ++i) tt[i] = 0.f;
      for (int w = 0; w < WG; ++w) {
        const float4 v4 = *reinterpret_cast<const float4*>(rs + w * kRB);
        tt[0] += v4.x; tt[1] += v4.y; tt[2] += v4.z; tt[3] += v4.w;
      }
      parity ^= 1;
    }
    if (gl == 0) {
#pragma unroll
      for (int i = 0; i < kRB; ++i)
        if (r0 + i < mb) {
          ttil_s[r0 + i] = tt[i];
          sacc += (double)tt[i] * (double)tt[i];
        }
    }
#pragma unroll
    for (int i = 0; i < kRB; ++i)
#pragma unroll
      for (int v = 0; v < NV; ++v) axpy4(q[v], x[i][v], tt[i]);
  }
#pragma unroll
  for (int v = 0; v < NV; ++v) *reinterpret_cast<float4*>(qs + (size_t)g * ldr + 4 * (gl + GT * v)) = q[v];
  if (gl == 0) sgrp[g] = sacc;
  __syncthreads();
}

// Combine the NG group partials and publish this CTA's partial raw loads (fixed order).
__device__ __forceinline__ void publish_q(const FusedParams& prm, const float* qs, float* qpart_row) {
  const int NG = kThreads / prm.GT, ldr = prm.ldr;
  for (int c = threadIdx.x * 4; c < ldr; c += kThreads * 4) {
    float4 a = *reinterpret_cast<const float4*>(qs + c);
    for (int g = 1; g < NG; ++g) {
      const float4 b = *reinterpret_cast<const float4*>(qs + (size_t)g * ldr + c);
      a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w;
    }
    *reinterpret_cast<float4*>(qpart_row + c) = a;
  }
}

// out_s[j] = sum_{b < nparts} part[b*stride + j] (float partials, fp64 sums, fixed order), j < count.
__device__ __forceinline__ void reduce_fparts(double* out_s, const float* part, int count, int nparts, int stride,
                                              double* scr) {
  for (int j0 = 0; j0 < count; j0 += kThreads) {
    const int cnt = min(count - j0, kThreads);
    const int cp = (cnt + 31) & ~31;
    int nsub = kThreads / cp;
    if (nsub > nparts) nsub = nparts;
    const int sub = threadIdx.x / cp, j = threadIdx.x - sub * cp;
    double v = 0.0;
    if (sub < nsub && j < cnt) {
      const float* src = part + j0 + j;
#pragma unroll 4
      for (int b = sub; b < nparts; b += nsub) v += (double)ld_cg(src + (size_t)b * stride);
    }
    __syncthreads();
    if (sub < nsub) scr[sub * cp + j] = v;
    __syncthreads();
    if (threadIdx.x < cnt) {
      double s = 0.0;
      for (int q = 0; q < nsub; ++q) s += scr[q * cp + threadIdx.x];
      out_s[j0 + threadIdx.x] = s;
    }
    __syncthreads();
  }
}

template <int NV, bool RESIDENT>
__global__ void __launch_bounds__(kThreads, 1) pca_fused_kernel(const FusedParams prm) {
  extern __shared__ __align__(16) unsigned char smem[];
  float* p_s = reinterpret_cast<float*>(smem + prm.off_p);        // ldr: current unit loads p
  float* pdef_s = reinterpret_cast<float*>(smem + prm.off_pdef);  // ldr: loads of the previous component
  float* ttil_s = reinterpret_cast<float*>(smem + prm.off_ttil);  // Mb : t0 / t~ rows of this CTA
  float* d_s = reinterpret_cast<float*>(smem + prm.off_d);        // Mb : pending deflation vector rows
  float* qs = reinterpret_cast<float*>(smem + prm.off_qs);        // NG x ldr group partials
  float* red_s = reinterpret_cast<float*>(smem + prm.off_red);    // 2 x kWarps x kRB
  double* sgrp = reinterpret_cast<double*>(smem + prm.off_sgrp);  // NG
  double* B_s = reinterpret_cast<double*>(smem + prm.off_B);      // Kpad
  double* A_s = reinterpret_cast<double*>(smem + prm.off_A);      // Kpad
  double* scr = reinterpret_cast<double*>(smem + prm.off_scr);    // kThreads
  double* praw_s = reinterpret_cast<double*>(smem + prm.off_praw);// Ns: p~ / p^ slice of this owner
  float* lam_s = reinterpret_cast<float*>(smem + prm.off_lam);    // Kpad
  float* slab = reinterpret_cast<float*>(smem + prm.off_slab);    // resident: Mb x ldr

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int b = blockIdx.x;
  const long long M = prm.M;
  const int N = prm.N, K = prm.K, G = prm.G, ldr = prm.ldr, Kpad = prm.Kpad;
  const int NG = kThreads / prm.GT;
  const bool gs = prm.algo == 1;
  const long long m0 = (long long)b * prm.Mb;
  const int mb = (int)max(0LL, min((long long)prm.Mb, M - m0));
  const int n0 = b * prm.Ns;
  const int ns = max(0, min(prm.Ns, N - n0));
  unsigned long long bar_target = 0;
  unsigned sweep_no = 0;                                   // parity selects the exchange buffers
  int tn = 0;                                              // trace records written (thread 0 of CTA 0)

  float* Rb = prm.Rrm + (size_t)m0 * ldr;
  float* Tb = prm.T + m0;

  for (int i = tid; i < prm.Mb; i += kThreads) d_s[i] = 0.f;
  for (int n = tid; n < ldr; n += kThreads) { p_s[n] = 0.f; pdef_s[n] = 0.f; }
  __syncthreads();

  for (int k = 0; k < K; ++k) {
    const bool gsk = gs && k > 0;
    trace_mark(prm, tn, TR_COMPONENT);
    // ---- S1: t0 <- column k of the deflated residual (reading C6) ----
    for (int i = tid; i < mb; i += kThreads) {
      float r;
      if (RESIDENT && k > 0) r = slab[(size_t)i * ldr + k];
      else r = ld_cg(Rb + (size_t)i * ldr + k);
      ttil_s[i] = fmaf(-d_s[i], pdef_s[k], r);
    }
    __syncthreads();
    // ---- LOADS sweep: pending deflation (S9) + q = R^T t0 (S2) ----
    if constexpr (RESIDENT) {
      if (k == 0) sweep_loads<NV, SRC_GLOBAL, DST_SLAB, false, true>(prm, Rb, slab, mb, ttil_s, d_s, pdef_s, qs);
      else        sweep_loads<NV, SRC_SLAB, DST_SLAB, true, true>(prm, Rb, slab, mb, ttil_s, d_s, pdef_s, qs);
    } else {
      if (k == 0) sweep_loads<NV, SRC_GLOBAL, DST_NONE, false, true>(prm, Rb, slab, mb, ttil_s, d_s, pdef_s, qs);
      else        sweep_loads<NV, SRC_GLOBAL, DST_GLOBAL, true, true>(prm, Rb, slab, mb, ttil_s, d_s, pdef_s, qs);
    }
    {
      const unsigned buf = sweep_no & 1u;
      publish_q(prm, qs, prm.Qpart + ((size_t)buf * G + b) * ldr);
      double s = 0.0;
      for (int i = tid; i < mb; i += kThreads) { const double v = (double)ttil_s[i]; s += v * v; }
      s = block_sum(s, scr);
      if (tid == 0) prm.Spart[(size_t)buf * G + b] = s;
    }
    trace_mark(prm, tn, TR_LOADS_DONE);

    double lam = 0.0, lam_new = 0.0;
    int it = 0;
    bool degenerate = false;
    bool first = true;
    for (;;) {
      const unsigned buf = sweep_no & 1u;
      const float* Qp = prm.Qpart + (size_t)buf * G * ldr;
      grid_barrier(prm.bar, bar_target, G);                                   // ---- X1 ----
      trace_mark(prm, tn, TR_X1);
      const double s = sum_parts(prm.Spart + (size_t)buf * G, G, scr);
      bool done = false;
      if (first) {
        if (!(s > 0.0)) { degenerate = true; break; }                         // zero start column (C7)
      } else {
        double bb = 0.0;
        if (gsk) {                                                            // B = V_(k)^T t~
          reduce_fparts(B_s, prm.Bpart + (size_t)buf * G * Kpad, k, G, Kpad, scr);
          double v = 0.0;
          for (int j = tid; j < k; j += kThreads) v += B_s[j] * B_s[j];
          bb = block_sum(v, scr);
        }
        const double l2 = s - bb;                                             // |t~ - V B|^2, V orthonormal
        if (!(l2 > 0.0)) { degenerate = true; break; }                        // reading C7
        lam_new = sqrt(l2);                                                   // S7
        // S8: listings' strict relative test (reading C3)
        done = (fabs(lam - lam_new) < prm.eps * lam_new) || (it >= prm.max_iter);
        if (!done) lam = lam_new;
      }
      trace_mark(prm, tn, TR_TEST);
      // ---- owners: q_S = sum of the G partials, fixed order, fp64 ----
      const bool need_q = !done || (gs && k + 1 < K);                         // finalize needs q only for W_k
      if (ns > 0 && need_q) {
        const int nsub = min(kThreads / ns, G);
        const int sub = tid / ns, i = tid - sub * ns;
        double v = 0.0;
        if (sub < nsub)
          for (int bq = sub; bq < G; bq += nsub) v += (double)ld_cg(Qp + (size_t)bq * ldr + n0 + i);
        if (sub < nsub) scr[sub * ns + i] = v;
        __syncthreads();
        if (tid < ns) {
          double a = 0.0;
          for (int q = 0; q < nsub; ++q) a += scr[q * ns + tid];
          praw_s[tid] = a;
        }
        __syncthreads();
        if (gsk && !first) {                                                  // p~ = q - W B
          const int nsub2 = kThreads / ns;
          const int sub2 = tid / ns, i2 = tid - sub2 * ns;
          double c = 0.0;
          if (sub2 < nsub2) {
            const float* wr = prm.W + (size_t)(n0 + i2) * Kpad;
            for (int j = sub2; j < k; j += nsub2) c += (double)ld_cg(wr + j) * B_s[j];
            scr[sub2 * ns + i2] = c;
          }
          __syncthreads();
          if (tid < ns) {
            double a = 0.0;
            for (int q = 0; q < nsub2; ++q) a += scr[q * ns + tid];
            praw_s[tid] -= a;
          }
          __syncthreads();
        }
      }
      if (done) break;
      trace_mark(prm, tn, TR_QSLICE);

      if (gsk) {
        // ---- S3: A-partials a_S[j] = sum_{n in S} P[n,j] p~[n] ----
        if (ns > 0) {
          for (int j = tid; j < k; j += kThreads) {
            const float* pj = prm.P + (size_t)j * N + n0;
            double a = 0.0;
            for (int i = 0; i < ns; ++i) a += (double)ld_cg(pj + i) * praw_s[i];
            prm.Apart[(size_t)b * Kpad + j] = (float)a;
          }
        }
        trace_mark(prm, tn, TR_APART);
        grid_barrier(prm.bar, bar_target, G);                                 // ---- X2 ----
        trace_mark(prm, tn, TR_X2);
        if (ns > 0) {
          reduce_fparts(A_s, prm.Apart, k, prm.Gs, Kpad, scr);
          // p^ = p~ - P_(k) A
          const int nsub = kThreads / ns;
          const int sub = tid / ns, i = tid - sub * ns;
          double c = 0.0;
          if (sub < nsub) {
            for (int j = sub; j < k; j += nsub) c += (double)ld_cg(prm.P + (size_t)j * N + n0 + i) * A_s[j];
            scr[sub * ns + i] = c;
          }
          __syncthreads();
          if (tid < ns) {
            double a = 0.0;
            for (int q = 0; q < nsub; ++q) a += scr[q * ns + tid];
            praw_s[tid] -= a;
          }
          __syncthreads();
        }
      }
      // ---- publish the p^ slice and its squared norm (S4, first half) ----
      if (ns > 0) {
        double q2 = 0.0;
        if (tid < ns) {
          const float v = (float)praw_s[tid];
          prm.pvec[n0 + tid] = v;
          q2 = (double)v * (double)v;
        }
        q2 = block_sum(q2, scr);
        if (tid == 0) prm.Npart[b] = q2;
      }
      trace_mark(prm, tn, TR_PHAT);
      grid_barrier(prm.bar, bar_target, G);                                   // ---- X3 ----
      trace_mark(prm, tn, TR_X3);
      const double pn2 = sum_parts(prm.Npart, prm.Gs, scr);
      if (!(pn2 > 0.0)) { degenerate = true; break; }                         // reading C7
      const float inv_pn = (float)(1.0 / sqrt(pn2));                          // p = p^/|p^|
      for (int n = tid; n < ldr; n += kThreads) p_s[n] = (n < N) ? ld_cg(prm.pvec + n) * inv_pn : 0.f;
      __syncthreads();
      first = false;
      trace_mark(prm, tn, TR_PREADY);
      // ---- FUSED sweep: t~ = R p (S5), q = R^T t~, s = |t~|^2 ----
      ++sweep_no;
      ++it;
      {
        const unsigned nbuf = sweep_no & 1u;
        const bool rev = (sweep_no & 1u) != 0;
        if constexpr (RESIDENT) sweep_fused<NV, SRC_SLAB>(prm, Rb, slab, mb, p_s, ttil_s, qs, red_s, sgrp, false);
        else                    sweep_fused<NV, SRC_GLOBAL>(prm, Rb, slab, mb, p_s, ttil_s, qs, red_s, sgrp, rev);
        trace_mark(prm, tn, TR_SWEEP);
        publish_q(prm, qs, prm.Qpart + ((size_t)nbuf * G + b) * ldr);
        if (tid == 0) {
          double a = 0.0;
          for (int g = 0; g < NG; ++g) a += sgrp[g];
          prm.Spart[(size_t)nbuf * G + b] = a;
        }
        if (gsk) {                                                            // S6: B-partials V^T t~
          float* bp = prm.Bpart + ((size_t)nbuf * G + b) * Kpad;
          for (int j = w; j < k; j += kWarps) {
            const float* vj = Tb + (size_t)j * M;
            float a = 0.f;
            for (int i = lane; i < mb; i += 32) a = fmaf(ld_cg(vj + i), ttil_s[i], a);
            const double sj = warp_sum((double)a);
            if (lane == 0) bp[j] = (float)sj;
          }
        }
        trace_mark(prm, tn, TR_PUBLISHED);
      }
    }

    // ---- component done ----
    if (degenerate) {
      for (int i = tid; i < mb; i += kThreads) { Tb[(size_t)k * M + i] = 0.f; d_s[i] = 0.f; }
      if (tid < ns) {
        prm.P[(size_t)k * N + n0 + tid] = 0.f;
        prm.W[(size_t)(n0 + tid) * Kpad + k] = 0.f;
      }
      for (int n = tid; n < ldr; n += kThreads) pdef_s[n] = 0.f;
      if (b == 0 && tid == 0) { prm.lambda[k] = 0.f; prm.iters[k] = 0; }
      if (tid == 0) lam_s[k] = 0.f;
    } else {
      const float lamf = (float)lam_new;
      const float inv = (float)(1.0 / lam_new);
      // t = t~ - V_(k) B;  GS-PCA: v = t/lambda'
      for (int i = tid; i < mb; i += kThreads) {
        float t = ttil_s[i];
        if (gsk) {
          float corr = 0.f;
          for (int j = 0; j < k; ++j) corr = fmaf(ld_cg(Tb + (size_t)j * M + i), (float)B_s[j], corr);
          t -= corr;
        }
        d_s[i] = t;                                                           // R -= lambda v p^T  /  R -= t p^T
        Tb[(size_t)k * M + i] = gs ? t * inv : t;
      }
      if (tid < ns) {
        const float pk = p_s[n0 + tid];
        prm.P[(size_t)k * N + n0 + tid] = pk;
        if (gs && k + 1 < K)                                                  // W_k = R_(k+1)^T v_k
          prm.W[(size_t)(n0 + tid) * Kpad + k] = (float)(praw_s[tid] / lam_new - lam_new * (double)pk);
      }
      for (int n = tid; n < ldr; n += kThreads) pdef_s[n] = p_s[n];
      if (b == 0 && tid == 0) { prm.lambda[k] = lamf; prm.iters[k] = it; }
      if (tid == 0) lam_s[k] = lamf;
    }
    ++sweep_no;                                                               // next LOADS sweep takes the other buffers
    __syncthreads();
    trace_mark(prm, tn, TR_FINAL);
  }
  if (prm.trace_cap > 0 && b == 0 && tid == 0) prm.trace[0] = (unsigned long long)tn;

  // resident: hand the slab back (the last deflation is applied by pca_transpose_out_kernel)
  if constexpr (RESIDENT) sweep_loads<NV, SRC_SLAB, DST_GLOBAL, false, false>(prm, Rb, slab, mb, ttil_s, d_s, pdef_s, qs);
  // ---- S10: GS-PCA  T <- V Lambda ----
  if (gs) {
    __syncthreads();
    for (int kk = 0; kk < K; ++kk) {
      const float l = lam_s[kk];
      for (int i = tid; i < mb; i += kThreads) Tb[(size_t)kk * M + i] *= l;
    }
  }
}

// ------------------------------------------------------------------------------------ transposes
// Rrm[m][n] = X[n*M + m] for n < N, 0 for N <= n < ldr                      (R <- X)
__global__ void __launch_bounds__(256) pca_transpose_in_kernel(const float* __restrict__ X, float* __restrict__ Rrm,
                                                               long long M, int N, int ldr) {
  __shared__ float tile[32][33];
  const long long mt = (long long)blockIdx.x * 32;
  const int nt = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;          // 32 x 8
#pragma unroll
  for (int j = ty; j < 32; j += 8) {
    const int n = nt + j;
    const long long m = mt + tx;
    tile[j][tx] = (n < N && m < M) ? __ldcg(X + (size_t)n * M + m) : 0.f;
  }
  __syncthreads();
#pragma unroll
  for (int j = ty; j < 32; j += 8) {
    const long long m = mt + j;
    const int n = nt + tx;
    if (m < M && n < ldr) Rrm[(size_t)m * ldr + n] = tile[tx][j];
  }
}

// Rout[n*M + m] = Rrm[m][n] - d[m]*p[n]: the residual of eq. (4) in the ABI's column-major layout,
// with the last component's deflation (d = T[:,K-1] after the epilogue, p = P[:,K-1]) applied.
__global__ void __launch_bounds__(256) pca_transpose_out_kernel(const float* __restrict__ Rrm, float* __restrict__ Rout,
                                                                const float* __restrict__ d, const float* __restrict__ p,
                                                                long long M, int N, int ldr) {
  __shared__ float tile[32][33];
  const long long mt = (long long)blockIdx.x * 32;
  const int nt = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
  for (int j = ty; j < 32; j += 8) {
    const long long m = mt + j;
    const int n = nt + tx;
    float v = 0.f;
    if (m < M && n < N) v = fmaf(-__ldcg(d + m), __ldcg(p + n), __ldcg(Rrm + (size_t)m * ldr + n));
    tile[j][tx] = v;
  }
  __syncthreads();
#pragma unroll
  for (int j = ty; j < 32; j += 8) {
    const int n = nt + j;
    const long long m = mt + tx;
    if (n < N && m < M) Rout[(size_t)n * M + m] = tile[tx][j];
  }
}

}  // namespace pca
