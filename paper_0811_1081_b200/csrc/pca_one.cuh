// =====================================================================================
// pca_one.cuh -- one-CTA solve kernel for matrices that fit in the register file of ONE SM
// (M <= (512/GT)*7 rows with GT = pow2 >= N/8 <= 64 threads per row; BASELINE.json config 1).
//
// Same rotated single-sweep iteration as pca_reg.cuh (t~ = R p and q = R^T t~ from the rows held in
// registers; scores-side projection folded into the loads through W = R^T V_(k); loads-side projection
// on the actual vector; PAPER.md:1016-1038 / :555-568), but with nothing to exchange: every reduction
// is a shuffle tree plus a block barrier, the whole loading panels P and W sit in shared memory, and a
// pass is the sweep plus five short phases.  The latency-bound end of the path (SURVEY.md section 8(d):
// "cfg 1: single-SM latency bound; report components/s and us/iteration").
// =====================================================================================
#pragma once
#include "pca_reg.cuh"

namespace pca {

struct OneParams {
  float* Rrm;            // M x ldr row-major residual (workspace): read once, written once
  float* T;              // M x K col-major
  float* P;              // N x K col-major
  float* lambda;         // K
  int* iters;            // K
  int M, N, K;
  double eps;
  int max_iter;
  int algo;              // 0 NIPALS, 1 GS
  int test_mode;         // 0 relative (listings), 1 absolute (text): pca_stagnated()
  int stag2;             // reading C4b: also compare lambda' with the value two passes back (PCA_OPT_STAGNATION)
  int out_svd;           // PCA_OPT_OUTPUT = 1: T holds the unit score vectors V (SVD triple V, U = P, Lambda)
  int ldr;               // 8*GT >= N
  int Kpad;
  // shared-memory carve-up (byte offsets)
  int off_p, off_ttil, off_d, off_qs, off_red, off_sgrp, off_q, off_B, off_A, off_scr, off_vb, off_pp, off_wp;
};

// The three reductions below are written for a compile-time number of lanes per item (PARTS = pow2 <= 32: shifts instead of
// divisions, unrolled shuffle trees) and dispatched on the run-time value, which is uniform over the CTA.  They are called
// by a ROLE: a set of whole warps (`nthr` threads, `rt` = the thread's index within the role), so that independent
// reductions of one phase run side by side on disjoint warps instead of one after the other on all of them.
template <int PARTS>
__device__ __forceinline__ double parts_sum(double a) {
#pragma unroll
  for (int o = PARTS >> 1; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  return a;
}
#define PCA_ONE_DISPATCH(parts, CALL) \
  switch (parts) {                    \
    case 1: { constexpr int PARTS = 1; CALL; } break;   \
    case 2: { constexpr int PARTS = 2; CALL; } break;   \
    case 4: { constexpr int PARTS = 4; CALL; } break;   \
    case 8: { constexpr int PARTS = 8; CALL; } break;   \
    case 16: { constexpr int PARTS = 16; CALL; } break; \
    default: { constexpr int PARTS = 32; CALL; } break; \
  }

// out[c] = sum_g in[g*ld + c] over ngroups, for c < n: `parts` consecutive lanes share a column (parts = pow2 <= 32),
// each sums every parts-th group in order, then a shuffle tree.  All threads of the CTA must call it.
template <int PARTS>
__device__ __forceinline__ void one_colsum_t(const float* in, int ld, int ngroups, int n, double* out, int tid, int nthr) {
  for (int c0 = 0; c0 < n; c0 += nthr / PARTS) {
    const int c = c0 + tid / PARTS, part = tid & (PARTS - 1);
    double a = 0.0;
    if (c < n) {
#pragma unroll 4
      for (int g = part; g < ngroups; g += PARTS) a += (double)in[(size_t)g * ld + c];
    }
    a = parts_sum<PARTS>(a);
    if (part == 0 && c < n) out[c] = a;
  }
}
__device__ __forceinline__ void one_colsum(const float* in, int ld, int ngroups, int n, int parts, double* out, int rt, int nthr) {
  PCA_ONE_DISPATCH(parts, one_colsum_t<PARTS>(in, ld, ngroups, n, out, rt, nthr))
}

// acc[i] = sum_{j<k} Mx[i*ld + j] * v[j] for i < n (row-major panel, odd row stride): `parts` lanes per row.
// f(i, value) is called by the first lane of each row.  All threads must call it.
template <int PARTS, typename F>
__device__ __forceinline__ void one_rowdot_t(const float* Mx, int ld, const double* v, int n, int k, F& f, int tid, int nthr) {
  for (int i0 = 0; i0 < n; i0 += nthr / PARTS) {
    const int i = i0 + tid / PARTS, part = tid & (PARTS - 1);
    double a = 0.0;
    if (i < n) {
#pragma unroll 4
      for (int j = part; j < k; j += PARTS) a += (double)Mx[(size_t)i * ld + j] * v[j];
    }
    a = parts_sum<PARTS>(a);
    if (part == 0 && i < n) f(i, a);
  }
}
template <typename F>
__device__ __forceinline__ void one_rowdot(const float* Mx, int ld, const double* v, int n, int k, int parts, F f, int rt, int nthr) {
  PCA_ONE_DISPATCH(parts, (one_rowdot_t<PARTS>(Mx, ld, v, n, k, f, rt, nthr)))
}

// acc[j] = sum_{i<n} Mx[i*ld + j] * v[i] for j < k (column sums of a row-major panel): `parts` lanes per column.
template <int PARTS, typename VT, typename F>
__device__ __forceinline__ void one_coldot_t(const float* Mx, int ld, const VT* v, int n, int k, F& f, int tid, int nthr) {
  for (int j0 = 0; j0 < k; j0 += nthr / PARTS) {
    const int j = j0 + tid / PARTS, part = tid & (PARTS - 1);
    double a = 0.0;
    if (j < k) {
#pragma unroll 4
      for (int i = part; i < n; i += PARTS) a += (double)Mx[(size_t)i * ld + j] * (double)v[i];
    }
    a = parts_sum<PARTS>(a);
    if (part == 0 && j < k) f(j, a);
  }
}
template <typename VT, typename F>
__device__ __forceinline__ void one_coldot(const float* Mx, int ld, const VT* v, int n, int k, int parts, F f, int rt, int nthr) {
  PCA_ONE_DISPATCH(parts, (one_coldot_t<PARTS, VT>(Mx, ld, v, n, k, f, rt, nthr)))
}

__device__ __forceinline__ int one_parts(int n, int nthr = kThreads) {   // lanes per item so that n items keep nthr threads busy: pow2 in [1, 32]
  int p = 32;
  while (p > 1 && n * p > nthr) p >>= 1;
  return p;
}

template <int GT, int RPT>
__global__ void __launch_bounds__(kThreads, 1) pca_one_kernel(const OneParams prm) {
  extern __shared__ __align__(16) unsigned char smem[];
  constexpr int NV = 2, NG = kThreads / GT;
  constexpr int NGQ = GT < 32 ? kWarps : NG;                       // rows of qs: the row groups of a warp pre-add their partial q (reg_sweep_*<..., WPRE>)
  float* p_s = reinterpret_cast<float*>(smem + prm.off_p);        // ldr: orthogonalised loads p^ of the last sweep
  float* ttil_s = reinterpret_cast<float*>(smem + prm.off_ttil);  // NG*RPT: t0 / t~
  float* d_s = reinterpret_cast<float*>(smem + prm.off_d);        // NG*RPT: deflation vector
  float* qs = reinterpret_cast<float*>(smem + prm.off_qs);        // NG x ldr group partials of q
  float* red_s = reinterpret_cast<float*>(smem + prm.off_red);    // kThreads
  double* sgrp = reinterpret_cast<double*>(smem + prm.off_sgrp);  // NG
  double* q_s = reinterpret_cast<double*>(smem + prm.off_q);      // ldr: q -> p~ -> p^ (fp64)
  double* B_s = reinterpret_cast<double*>(smem + prm.off_B);      // Kpad
  double* A_s = reinterpret_cast<double*>(smem + prm.off_A);      // Kpad
  double* scr = reinterpret_cast<double*>(smem + prm.off_scr);    // kThreads (block_sum) ; ctl at the end
  double* ctl_s = scr + kThreads - 8;                             // [0] |t~|^2 [1] lambda' [2] decision
  float* Vb = reinterpret_cast<float*>(smem + prm.off_vb);        // NG*RPT x KV: unit scores
  float* Pp = reinterpret_cast<float*>(smem + prm.off_pp);        // ldr x KV: loadings P_(k)
  float* Wp = reinterpret_cast<float*>(smem + prm.off_wp);        // ldr x KV: W = R^T V_(k)

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int g = tid / GT, gl = tid - g * GT;
  const int M = prm.M, N = prm.N, K = prm.K, ldr = prm.ldr, KV = prm.Kpad | 1;
  const int mb = M;
  const bool gs = prm.algo == 1;
  float* Rb = prm.Rrm;

  RowBlock<NV, RPT, 0> Rr;                                         // R <- X, in registers
  Rr.sm = nullptr; Rr.rstride = 0; Rr.vstride = 0;
#pragma unroll
  for (int i = 0; i < RPT; ++i) {
    const int r = g * RPT + i;
#pragma unroll
    for (int v = 0; v < NV; ++v)
      Rr.r[i][v] = (r < mb) ? ld_stream4(Rb + (size_t)r * ldr + 4 * (gl + GT * v)) : make_float4(0.f, 0.f, 0.f, 0.f);
  }
  for (int i = tid; i < NG * RPT; i += kThreads) { d_s[i] = 0.f; ttil_s[i] = 0.f; }
  for (int n = tid; n < ldr; n += kThreads) { p_s[n] = 0.f; q_s[n] = 0.0; }
  __syncthreads();
  const int pq = one_parts(ldr);                                   // lanes per column in the N-side phases run by all warps
  // Roles of the two phases with independent work (whole warps each; kWarps = 16): the last warp takes the scalar chain
  // (|t~|^2, then lambda' and the test); with Gram-Schmidt coefficients to form, warps 0-7 combine q while warps 8-14 form B.
  constexpr int kScalarWarp = kWarps - 1, kQWarpsB = 8;

  for (int k = 0; k < K; ++k) {
    const bool gsk = gs && k > 0;
    // ---- S1 + S2: t0 <- column k of the deflated residual; q = R^T t0 ----
    reg_sweep_loads<GT, NV, RPT, true>(Rr, k, ttil_s, qs, sgrp, ldr);
    double lam = 0.0, lam2 = 0.0, lam_new = 0.0;
    int it = 0;
    bool degenerate = false, first = true;
    float pscale = 0.f;
    const int pk2 = one_parts(k > 0 ? k : 1);
    for (;;) {
      const bool with_b = gsk && !first;
      // ---- q = sum of the group partials (fp64);  |t~|^2;  B = V_(k)^T t~ (S6) ----
      {
        const int wq = with_b ? kQWarpsB : kScalarWarp;
        if (w < wq) {
          one_colsum(qs, ldr, NGQ, ldr, one_parts(ldr, 32 * wq), q_s, tid, 32 * wq);
        } else if (w < kScalarWarp) {
          constexpr int nb = 32 * (kScalarWarp - kQWarpsB);
          one_coldot<float>(Vb, KV, ttil_s, mb, k, one_parts(k, nb), [&](int j, double a) { B_s[j] = a; }, tid - 32 * kQWarpsB, nb);
        } else {
          double s = 0.0;
          for (int gg = lane; gg < NG; gg += 32) s += sgrp[gg];
          s = warp_sum(s);
          if (lane == 0) ctl_s[0] = s;
        }
      }
      __syncthreads();
      // ---- S7 / S8 by the scalar warp;  p~ = q - W B by the others ----
      if (w == kScalarWarp) {
        const double s = ctl_s[0];
        int st = 0;
        double ln = 0.0;
        if (first) {
          if (!(s > 0.0)) st = 2;                                             // zero start column (C7)
        } else {
          double bb = 0.0;
          if (gsk) {
            for (int j = lane; j < k; j += 32) bb += B_s[j] * B_s[j];
            bb = warp_sum(bb);
          }
          const double l2 = s - bb;                                           // |t~ - V B|^2, V orthonormal
          if (!(l2 > 0.0)) st = 2;
          else {
            ln = fast_sqrt(l2);                                               // S7
            // S8: the listings' strict relative test (readings C3, C4b)
            if (pca_stagnated(lam, lam2, ln, prm.eps, prm.test_mode, prm.stag2) || (it >= prm.max_iter)) st = 1;
          }
        }
        if (lane == 0) { ctl_s[1] = ln; reinterpret_cast<int*>(ctl_s + 2)[0] = st; }
      } else if (with_b) {
        constexpr int nw = 32 * kScalarWarp;
        one_rowdot(Wp, KV, B_s, N, k, one_parts(N, nw), [&](int c, double a) { q_s[c] -= a; }, tid, nw);
      }
      __syncthreads();
      const int st = reinterpret_cast<const int*>(ctl_s + 2)[0];
      if (st == 2) { degenerate = true; break; }
      if (!first) {
        lam_new = ctl_s[1];
        if (st == 1) break;                                                   // q_s = R^T t, p_s = the loads of the last sweep
        lam2 = lam;
        lam = lam_new;
      }
      // ---- S3: A = P_(k)^T p~ ;  p^ = p~ - P_(k) A;  S4: p = p^ / |p^| (the scale is applied
      //      by the sweep).  p_s[N..ldr) stays zero from the start of the kernel. ----
      if (gsk) {
        one_coldot<double>(Pp, KV, q_s, N, k, pk2, [&](int j, double a) { A_s[j] = a; }, tid, kThreads);
        __syncthreads();
      }
      if (gsk) {
        one_rowdot(Pp, KV, A_s, N, k, pq, [&](int c, double a) {
          const double x = q_s[c] - a;
          q_s[c] = x;
          p_s[c] = (float)x;
        }, tid, kThreads);
      } else {
        for (int c = tid; c < N; c += kThreads) p_s[c] = (float)q_s[c];
      }
      __syncthreads();
      // |p^|^2 of the fp32 loads the sweep will use: every warp forms it itself from p_s (same order in every warp), which
      // costs one shuffle tree instead of two trees and a second barrier
      double n2 = 0.0;
      for (int c = lane; c < N; c += 32) { const double v = (double)p_s[c]; n2 += v * v; }
      n2 = warp_sum(n2);
      pscale = (n2 > 0.0) ? (float)rsqrt(n2) : 0.f;
      if (!(pscale > 0.f)) { degenerate = true; break; }                      // reading C7
      first = false;
      ++it;
      // ---- FUSED sweep: t~ = R p (S5), q = R^T t~ (S2 of the next pass) ----
      reg_sweep_fused<GT, NV, RPT, true>(Rr, p_s, pscale, ttil_s, qs, red_s, sgrp, ldr);
    }

    if (degenerate) {
      for (int i = tid; i < NG * RPT; i += kThreads) {
        if (i < mb) prm.T[(size_t)k * M + i] = 0.f;
        if (gs) Vb[(size_t)i * KV + k] = 0.f;
      }
      for (int c = tid; c < ldr; c += kThreads) {
        if (c < N) prm.P[(size_t)k * N + c] = 0.f;
        if (gs) { Pp[(size_t)c * KV + k] = 0.f; Wp[(size_t)c * KV + k] = 0.f; }
      }
      if (tid == 0) { prm.lambda[k] = 0.f; prm.iters[k] = 0; }
      __syncthreads();
    } else {
      const float inv = (float)(1.0 / lam_new);
      // t = t~ - V_(k) B;  v = t/lambda';  T[:,k] = lambda' v = t (:87,:1037)
      one_rowdot(Vb, KV, B_s, mb, gsk ? k : 0, one_parts(mb), [&](int r, double a) {
        const float t = ttil_s[r] - (float)a;
        d_s[r] = t;
        prm.T[(size_t)k * M + r] = prm.out_svd ? t * inv : t;                 // SVD output: the unit vector v
        if (gs) Vb[(size_t)r * KV + k] = t * inv;
      }, tid, kThreads);
      for (int c = tid; c < ldr; c += kThreads) {
        const float pk = p_s[c] * pscale;
        if (c < N) prm.P[(size_t)k * N + c] = pk;
        if (gs) {
          Pp[(size_t)c * KV + k] = pk;
          if (k + 1 < K) Wp[(size_t)c * KV + k] = (float)(q_s[c] / lam_new - lam_new * (double)pk);   // W_k = R_(k+1)^T v_k
        }
      }
      if (tid == 0) { prm.lambda[k] = (float)lam_new; prm.iters[k] = it; }
      __syncthreads();
      // ---- S9: rank-1 deflation in registers (eq. 3) ----
      float4 p4[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        p4[v] = *reinterpret_cast<const float4*>(p_s + 4 * (gl + GT * v));
        p4[v].x *= pscale; p4[v].y *= pscale; p4[v].z *= pscale; p4[v].w *= pscale;
      }
#pragma unroll
      for (int i = 0; i < RPT; ++i) {
        const float dr = -d_s[g * RPT + i];
#pragma unroll
        for (int v = 0; v < NV; ++v) axpy4(Rr.r[i][v], p4[v], dr);
      }
    }
  }
  // ---- the residual of eq. (4), back to the row-major workspace ----
#pragma unroll
  for (int i = 0; i < RPT; ++i) {
    const int r = g * RPT + i;
    if (r < mb) {
#pragma unroll
      for (int v = 0; v < NV; ++v) *reinterpret_cast<float4*>(Rb + (size_t)r * ldr + 4 * (gl + GT * v)) = Rr.r[i][v];
    }
  }
}

typedef void (*one_kernel_t)(const OneParams);
one_kernel_t one_kernel_lookup(int GT, int RPT);       // defined in pca_reg_inst.cu (parts 0 and 1), nullptr if absent

}  // namespace pca
