// =====================================================================================
// pca_solve.cuh -- the persistent, grid-synchronised solve kernel: all K components, all inner
// passes, convergence tested on the device (no host round-trip), one launch per pca_run.
//
// Per component k (statement order of PAPER.md:555-568 / :1016-1038):
//   S1  t <- column k of the deflated residual
//   loop (at most max_iter passes):
//     Ph1  S2  partial loads  pp_b = R_b^T t_b                (first pass of a component also
//              applies the previous component's deflation S9, or the copy R <- X for k = 0)
//     ---- grid barrier ----
//     Ph2      column-slice owners sum the G partials -> p~ ;  GS-PCA: A-partials  P_(k)^T p~   (S3)
//     ---- grid barrier (GS-PCA, k > 0) ----
//     Ph3      GS-PCA: A = sum of partials;  p^ = p~ - P_(k) A ;  ||p^||^2 partials            (S3, S4)
//     ---- grid barrier ----
//     Ph4  S4  p = p^ / ||p^|| ;  S5  t_b = R_b p ;  GS-PCA: B-partials V_(k)^T t               (S6)
//     ---- grid barrier (GS-PCA, k > 0) ----
//     Ph5      GS-PCA: B = sum of partials;  t_b -= V_b B ;  ||t||^2 partials                   (S6, S7)
//     ---- grid barrier ----
//     Ph6  S7  lambda' = ||t|| ;  GS-PCA: t /= lambda' ;  S8 test |lambda - lambda'| < eps lambda'
//   store T[:,k], P[:,k], lambda[k], iters[k];  d <- (GS ? lambda' v : t) for the next deflation
// after the last component: final deflation (R of eq. 4) and GS-PCA's T <- V Lambda (S10).
// =====================================================================================
#pragma once
#include "pca_device.cuh"

namespace pca {

// T = float: fp32 storage (BASELINE.json); T = double: the paper's native precision, everything in fp64
template <typename T>
struct SolveParamsT {
  const T* X;        // M x N centred input (never written)
  T* R;              // M x N residual workspace
  T* Tm;             // M x K
  T* P;              // N x K
  T* lambda;         // K
  int* iters;            // K
  long long M, N;
  int K;
  double eps;
  int max_iter;
  int algo;              // 0 NIPALS, 1 GS
  int test_mode;         // 0 relative (listings), 1 absolute (text): pca_stagnated()
  int stag2;             // reading C4b: also compare lambda' with the value two passes back (PCA_OPT_STAGNATION)
  int out_svd;           // PCA_OPT_OUTPUT = 1: T holds the unit score vectors V (SVD triple V, U = P, Lambda)
  int gs_passes;         // classical Gram-Schmidt projections per side per inner pass: 1 (the listings), 2 = CGS2 ("applying it
                         // iteratively"; PCA_OPT_GS_PASSES)
  int G;                 // CTAs
  int Mb;                // rows per CTA (uniform; last CTAs may own fewer / none)
  int Ns;                // columns per slice owner (multiple of 4)
  int Gs;                // number of slice owners = ceil(N / Ns) <= G
  int slab_ld;           // resident path: column stride of the SMEM slab (floats)
  int Npad;              // row stride of Ppart (floats)
  int Kpad;              // row stride of Apart / Bpart (doubles)
  T* Ppart;          // [G][Npad]   partial loads
  double* Apart;         // [2][Gs][Kpad]  partial A (loads-side GS coefficients), one buffer per CGS projection
  double* Bpart;         // [2][G][Kpad]   partial B (scores-side GS coefficients)
  T* pvec;           // [Npad]      p^ (orthogonalised, not yet normalised)
  double* qpart;         // [Gs]        ||p^||^2 partials
  double* spart;         // [G]         ||t||^2 partials
  unsigned long long* bar;  // grid barrier counter (zeroed before launch)
  // shared memory carve-up (bytes from the start of dynamic smem), computed by the host plan
  int off_t, off_d, off_p, off_slice, off_coef, off_lam, off_scr, off_red, off_slab;
};
typedef SolveParamsT<float> SolveParams;

template <typename T, bool RESIDENT, int VEC, int TR, int RC>
__device__ __forceinline__ void pca_solve_body(const SolveParamsT<T>& prm) {
  extern __shared__ __align__(16) unsigned char smem[];
  T* t_s = reinterpret_cast<T*>(smem + prm.off_t);          // Mb: this CTA's rows of t / v
  T* d_s = reinterpret_cast<T*>(smem + prm.off_d);          // Mb: deflation vector rows
  T* p_s = reinterpret_cast<T*>(smem + prm.off_p);          // N : full loads vector
  T* slice_s = reinterpret_cast<T*>(smem + prm.off_slice);  // Ns: this CTA's slice of p~ / p^
  double* coef_s = reinterpret_cast<double*>(smem + prm.off_coef);  // K : A or B
  T* lam_s = reinterpret_cast<T*>(smem + prm.off_lam);      // K : lambda_k (GS final scaling)
  double* scr = reinterpret_cast<double*>(smem + prm.off_scr);      // kThreads doubles scratch
  T* red_s = reinterpret_cast<T*>(smem + prm.off_red);      // kWarps * CH floats
  T* slab = reinterpret_cast<T*>(smem + prm.off_slab);      // resident slab [N][slab_ld]

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int b = blockIdx.x;
  const long long M = prm.M;
  const int N = (int)prm.N, K = prm.K, G = prm.G;
  const bool gs = prm.algo == 1;
  const long long m0 = (long long)b * prm.Mb;
  const int mb = (int)max(0LL, min((long long)prm.Mb, M - m0));
  const int n0 = b * prm.Ns;
  const int ns = max(0, min(prm.Ns, N - n0));
  const int slab_ld = prm.slab_ld;
  unsigned long long bar_target = 0;

  const T* Xb = prm.X + m0;          // row-offset views (column stride M)
  T* Rb = prm.R + m0;
  T* Tb = prm.Tm + m0;
  T* my_part = prm.Ppart + (size_t)b * prm.Npad;

  for (int i = tid; i < prm.Mb; i += kThreads) d_s[i] = T(0);
  for (int n = tid; n < N; n += kThreads) p_s[n] = T(0);
  __syncthreads();

  for (int k = 0; k < K; ++k) {
    // ---- S1: t <- R^(k) of the deflated residual (reading C6) ----
    for (int i = tid; i < mb; i += kThreads) {
      T r;
      if (k == 0) r = ld_cg(Xb + i);                                   // R <- X not yet materialised
      else if constexpr (RESIDENT) r = slab[(size_t)k * slab_ld + i];
      else r = ld_cg(Rb + (size_t)k * M + i);
      t_s[i] = fma_t(-d_s[i], p_s[k], r);                               // pending deflation of comp k-1
    }
    __syncthreads();

    double lam = 0.0, lam2 = 0.0, lam_new = 0.0;
    int it = 0;
    bool degenerate = false;
    for (int j = 0; j < prm.max_iter; ++j) {
      // ---- Ph1: partial loads (S2), fused with deflation / copy on the first pass (S9, A2) ----
      if (j == 0) {
        if constexpr (RESIDENT) {
          if (k == 0) pass_t<T, VEC, TR, RC, SRC_GLOBAL, DST_SLAB, true, true>(Xb, nullptr, M, slab, slab_ld, mb, N, t_s, d_s, p_s, my_part);
          else        pass_t<T, VEC, TR, RC, SRC_SLAB, DST_SLAB, true, true>(nullptr, nullptr, M, slab, slab_ld, mb, N, t_s, d_s, p_s, my_part);
        } else {
          pass_t<T, VEC, TR, RC, SRC_GLOBAL, DST_GLOBAL, true, true>(k == 0 ? Xb : Rb, Rb, M, nullptr, 0, mb, N, t_s, d_s, p_s, my_part);
        }
      } else {
        if constexpr (RESIDENT) pass_t<T, VEC, TR, RC, SRC_SLAB, DST_NONE, false, true>(nullptr, nullptr, M, slab, slab_ld, mb, N, t_s, d_s, p_s, my_part);
        else                    pass_t<T, VEC, TR, RC, SRC_GLOBAL, DST_NONE, false, true>(Rb, nullptr, M, nullptr, 0, mb, N, t_s, d_s, p_s, my_part);
      }
      if (mb == 0) for (int n = tid; n < N; n += kThreads) my_part[n] = T(0);   // CTA without rows
      grid_barrier(prm.bar, bar_target, G);

      // ---- Ph2: slice owners reduce the G partials: p~[n] = sum_b pp_b[n] ----
      if (ns > 0) {
        const int nsub = min(kThreads / ns, G);
        const int sub = tid / ns, i = tid - sub * ns;
        double v = 0.0;
        if (sub < nsub)
          for (int bb = sub; bb < G; bb += nsub) v += (double)ld_cg(prm.Ppart + (size_t)bb * prm.Npad + n0 + i);
        if (sub < nsub) scr[sub * ns + i] = v;
        __syncthreads();
        if (tid < ns) {
          double s = 0.0;
          for (int q = 0; q < nsub; ++q) s += scr[q * ns + tid];
          slice_s[tid] = (T)s;
        }
        __syncthreads();
      }
      if (gs && k > 0) {
        for (int rep = 0; rep < prm.gs_passes; ++rep) {                  // CGS2: project a second time
          double* Apart = prm.Apart + (size_t)rep * prm.Gs * prm.Kpad;
          // ---- S3: A-partials  a_b[jj] = sum_{n in slice} P[n,jj] p~[n] ----
          if (ns > 0) {
            for (int jj = tid; jj < k; jj += kThreads) {
              const T* pj = prm.P + (size_t)jj * N + n0;
              double a = 0.0;
              for (int i = 0; i < ns; ++i) a += (double)ld_cg(pj + i) * (double)slice_s[i];
              Apart[(size_t)b * prm.Kpad + jj] = a;
            }
          }
          grid_barrier(prm.bar, bar_target, G);
          // ---- Ph3: A = sum of partials;  p^ = p~ - P_(k) A ----
          if (ns > 0) {
            reduce_coef_parts(coef_s, Apart, k, prm.Gs, prm.Kpad, scr);
            const int nsub = kThreads / ns;
            const int sub = tid / ns, i = tid - sub * ns;
            double v = 0.0;
            if (sub < nsub)
              for (int jj = sub; jj < k; jj += nsub) v += (double)ld_cg(prm.P + (size_t)jj * N + n0 + i) * coef_s[jj];
            __syncthreads();
            if (sub < nsub) scr[sub * ns + i] = v;
            __syncthreads();
            if (tid < ns) {
              double s = 0.0;
              for (int q = 0; q < nsub; ++q) s += scr[q * ns + tid];
              slice_s[tid] = (T)((double)slice_s[tid] - s);
            }
            __syncthreads();
          }
        }
      }
      // ---- S4 (first half): ||p^||^2 partial, publish the slice ----
      if (ns > 0) {
        double q = 0.0;
        if (tid < ns) {
          const T v = slice_s[tid];
          prm.pvec[n0 + tid] = v;
          q = (double)v * (double)v;
        }
        q = block_sum(q, scr);
        if (tid == 0) prm.qpart[b] = q;
      }
      grid_barrier(prm.bar, bar_target, G);

      // ---- Ph4: p = p^/||p^||;  S5: t = R p ----
      const double pn2 = sum_parts(prm.qpart, prm.Gs, scr);
      if (!(pn2 > 0.0)) { degenerate = true; break; }                 // reading C7 (uniform across CTAs)
      const T inv_pn = (T)(1.0 / sqrt(pn2));
      for (int n = tid; n < N; n += kThreads) p_s[n] = ld_cg(prm.pvec + n) * inv_pn;
      __syncthreads();
      if constexpr (RESIDENT) pass_n<T, VEC, TR, RC, SRC_SLAB>(nullptr, M, slab, slab_ld, mb, N, p_s, t_s, red_s);
      else                    pass_n<T, VEC, TR, RC, SRC_GLOBAL>(Rb, M, nullptr, 0, mb, N, p_s, t_s, red_s);

      if (gs && k > 0) {
        for (int rep = 0; rep < prm.gs_passes; ++rep) {                  // CGS2: project a second time
          double* Bpart = prm.Bpart + (size_t)rep * G * prm.Kpad;
          // ---- S6: B-partials  b_b[jj] = sum_{rows} V[m,jj] t[m] ----
          for (int jj = w; jj < k; jj += kWarps) {
            const T* vj = Tb + (size_t)jj * M;
            T a = T(0);
            for (int i = lane; i < mb; i += 32) a = fma_t(ld_cg(vj + i), t_s[i], a);
            const double s = warp_sum((double)a);
            if (lane == 0) Bpart[(size_t)b * prm.Kpad + jj] = s;
          }
          grid_barrier(prm.bar, bar_target, G);
          // ---- Ph5: B = sum of partials;  t -= V_(k) B ----
          reduce_coef_parts(coef_s, Bpart, k, G, prm.Kpad, scr);
          for (int i = tid; i < mb; i += kThreads) {
            T corr = T(0);
            for (int jj = 0; jj < k; ++jj) corr = fma_t(ld_cg(Tb + (size_t)jj * M + i), (T)coef_s[jj], corr);
            t_s[i] -= corr;
          }
          __syncthreads();
        }
      }
      // ---- S7: lambda' = ||t|| ----
      {
        double s = 0.0;
        for (int i = tid; i < mb; i += kThreads) { const double v = (double)t_s[i]; s += v * v; }
        s = block_sum(s, scr);
        if (tid == 0) prm.spart[b] = s;
      }
      grid_barrier(prm.bar, bar_target, G);
      const double l2 = sum_parts(prm.spart, G, scr);
      if (!(l2 > 0.0)) { degenerate = true; break; }                  // reading C7
      lam_new = sqrt(l2);
      if (gs) {                                                       // V^(k) <- V^(k)/lambda_k
        const T inv = (T)(1.0 / lam_new);
        for (int i = tid; i < mb; i += kThreads) t_s[i] *= inv;
        __syncthreads();
      }
      it = j + 1;
      // ---- S8: listings' strict relative test (reading C3) ----
      if (pca_stagnated(lam, lam2, lam_new, prm.eps, prm.test_mode, prm.stag2)) break;   // S8 (readings C3, C4b)
      lam2 = lam;
      lam = lam_new;
    }

    // ---- component done: store, and set up the pending deflation ----
    if (degenerate) {
      for (int i = tid; i < mb; i += kThreads) { Tb[(size_t)k * M + i] = 0.f; d_s[i] = T(0); t_s[i] = 0.f; }
      if (tid < ns) prm.P[(size_t)k * N + n0 + tid] = T(0);
      if (b == 0 && tid == 0) { prm.lambda[k] = T(0); prm.iters[k] = 0; }
      if (tid == 0) lam_s[k] = T(0);
    } else {
      const T lamf = (T)lam_new;
      const T tscale = (!gs && prm.out_svd) ? (T)(1.0 / lam_new) : T(1);   // SVD output of NIPALS-PCA: v = t/lambda
      for (int i = tid; i < mb; i += kThreads) {
        const T v = t_s[i];
        Tb[(size_t)k * M + i] = v * tscale;                           // GS-PCA: unit v until the final scaling
        d_s[i] = gs ? lamf * v : v;                                   // R -= lambda v p^T / R -= t p^T
      }
      if (tid < ns) prm.P[(size_t)k * N + n0 + tid] = p_s[n0 + tid];
      if (b == 0 && tid == 0) { prm.lambda[k] = lamf; prm.iters[k] = it; }
      if (tid == 0) lam_s[k] = lamf;
    }
    __syncthreads();
  }

  // ---- final deflation: the residual R of eq. (4) ----
  if constexpr (RESIDENT)
    pass_t<T, VEC, TR, RC, SRC_SLAB, DST_GLOBAL, true, false>(nullptr, Rb, M, slab, slab_ld, mb, N, t_s, d_s, p_s, my_part);
  else
    pass_t<T, VEC, TR, RC, SRC_GLOBAL, DST_GLOBAL, true, false>(Rb, Rb, M, nullptr, 0, mb, N, t_s, d_s, p_s, my_part);
  // ---- S10: GS-PCA  T <- V Lambda; skipped for the SVD output V, U, Lambda ----
  if (gs && !prm.out_svd) {
    __syncthreads();
    for (int kk = 0; kk < K; ++kk) {
      const T l = lam_s[kk];
      for (int i = tid; i < mb; i += kThreads) Tb[(size_t)kk * M + i] *= l;
    }
  }
}

template <bool RESIDENT, int VEC, int TR, int RC>
__global__ void __launch_bounds__(kThreads, 1) pca_solve_kernel(const SolveParams prm) {
  pca_solve_body<float, RESIDENT, VEC, TR, RC>(prm);
}
// fp64 storage and arithmetic throughout (the paper's precision): scalar lane mapping
static __global__ void __launch_bounds__(kThreads, 1) pca_solve_f64_kernel(const SolveParamsT<double> prm) {
  pca_solve_body<double, false, 1, 32, 4>(prm);
}

}  // namespace pca
