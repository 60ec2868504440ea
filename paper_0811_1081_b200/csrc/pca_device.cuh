// =====================================================================================
// pca_device.cuh -- device-side building blocks of the persistent PCA solve kernel (sm_100a).
//
// Data decomposition: the residual R (M x N, column-major, ld = M) is
// split into G ROW BLOCKS, one per CTA of a persistent cooperative kernel.  CTA b owns rows
// [b*Mb, b*Mb + mb).  With row ownership
//   * scores  t = R p        (S5) are LOCAL to the CTA given the full p;
//   * loads   p = R^T t      (S2) are per-CTA partial sums over its rows,
//                            combined across CTAs through a small L2-resident exchange buffer;
//   * deflation R -= d p^T   (S9) is LOCAL (d = the CTA's rows of t / lambda v).
// The slab of a CTA either lives in shared memory for the whole solve (resident path) or is
// streamed from HBM/L2 every pass (streaming path); both use the same lane mapping:
//   a warp covers CW = 32/TR columns at once, TR lanes along the rows of a column,
//   each lane holding RC row-vectors of VEC floats (VEC = 4 -> 128-bit loads).
// =====================================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pca {

constexpr int kThreads = 512;           // threads per CTA of the solve kernel
constexpr int kWarps = kThreads / 32;

enum { SRC_GLOBAL = 0, SRC_SLAB = 1 };
enum { DST_NONE = 0, DST_GLOBAL = 1, DST_SLAB = 2 };

// ------------------------------------------------------------------------------------ loads
// Exchange buffers and R are read with ld.global.cg (L2 only): other CTAs write the exchange
// buffers during the kernel, and the R stream has no L1 reuse.
__device__ __forceinline__ float ld_cg(const float* p) { return __ldcg(p); }
__device__ __forceinline__ double ld_cg(const double* p) { return __ldcg(p); }
__device__ __forceinline__ float4 ld_cg4(const float* p) {
  return __ldcg(reinterpret_cast<const float4*>(p));
}

// T = float (fp32 storage, the build's default) or double (the paper's native precision: VEC = 1)
__device__ __forceinline__ float fma_t(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_t(double a, double b, double c) { return fma(a, b, c); }

template <typename T, int VEC>
__device__ __forceinline__ void load_vec(T (&x)[VEC], const T* p) {
  if constexpr (VEC == 4 && sizeof(T) == 4) {
    const float4 v = ld_cg4(reinterpret_cast<const float*>(p));
    x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
  } else {
#pragma unroll
    for (int e = 0; e < VEC; ++e) x[e] = ld_cg(p + e);
  }
}
template <typename T, int VEC>
__device__ __forceinline__ void load_vec_smem(T (&x)[VEC], const T* p) {
  if constexpr (VEC == 4 && sizeof(T) == 4) {
    const float4 v = *reinterpret_cast<const float4*>(p);
    x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
  } else {
#pragma unroll
    for (int e = 0; e < VEC; ++e) x[e] = p[e];
  }
}
template <typename T, int VEC>
__device__ __forceinline__ void store_vec(T* p, const T (&x)[VEC]) {
  if constexpr (VEC == 4 && sizeof(T) == 4) {
    *reinterpret_cast<float4*>(p) = make_float4(x[0], x[1], x[2], x[3]);
  } else {
#pragma unroll
    for (int e = 0; e < VEC; ++e) p[e] = x[e];
  }
}

// ------------------------------------------------------------------------------------ grid barrier
// All G CTAs of the cooperative launch are co-resident.  Monotonic 64-bit arrival counter,
// zeroed by the host before the launch; `target` is each CTA's private count of expected arrivals.
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_add_u64(unsigned long long* p, unsigned long long v) {
  asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

__device__ __forceinline__ void grid_barrier(unsigned long long* ctr, unsigned long long& target, int G) {
  __syncthreads();
  if (G > 1) {
    target += (unsigned long long)G;
    if (threadIdx.x == 0) {
      __threadfence();
      red_release_add_u64(ctr, 1ULL);
      while (ld_acquire_u64(ctr) < target) { /* spin */ }
      __threadfence();
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------ convergence test (S8)
// mode 0: the listings' strict relative test |lambda - lambda'| < eps*lambda' (reading C3, default)
// mode 1: the text's / pseudo-code's absolute test |lambda' - lambda| <= eps
// lam = lambda of the previous pass (0 before the first), lam2 = of the one before (0 = none yet):
// reading C4b (stag2 != 0, PCA_OPT_STAGNATION = 1, the default): a period-2 limit cycle of lambda' in fp32 is stagnation
// too, so lambda' is also compared with the value two passes back.  stag2 == 0: the listing's / text's test alone.
// sqrt(x) and 1/x for a normal x > 0 from rsqrt(x) plus one Newton step (a few ulp at most).  sqrt() and the fp64 division are
// 300-cycle routines (measured on B200: sqrt 313, rsqrt 99 cycles of dependent latency) and lambda' = sqrt(.) sits on the serial
// per-pass chain of the convergence test that every CTA waits for.
__device__ __forceinline__ double fast_sqrt(double x) {
  const double r = rsqrt(x);
  const double y = x * r;
  return fma(fma(-y, y, x), 0.5 * r, y);
}
__device__ __forceinline__ double fast_rcp(double x) {
  const double r = rsqrt(x);
  const double y = r * r;
  return fma(fma(-x, y, 1.0), y, y);
}

__device__ __forceinline__ bool pca_stagnated(double lam, double lam2, double ln, double eps, int mode, int stag2) {
  const bool two = stag2 != 0 && lam2 > 0.0;
  if (mode == 1) return fabs(ln - lam) <= eps || (two && fabs(ln - lam2) <= eps);
  return fabs(lam - ln) < eps * ln || (two && fabs(lam2 - ln) < eps * ln);
}

// ------------------------------------------------------------------------------------ block reductions
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Sum of one double per thread over the CTA, returned to every thread.  Fixed order.
// scr: >= kWarps + 1 doubles of shared memory.
__device__ __forceinline__ double block_sum(double v, double* scr) {
  v = warp_sum(v);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  __syncthreads();                       // scr may still be read from a previous call
  if (lane == 0) scr[w] = v;
  __syncthreads();
  if (w == 0) {
    double s = (lane < kWarps) ? scr[lane] : 0.0;
    s = warp_sum(s);
    if (lane == 0) scr[kWarps] = s;
  }
  __syncthreads();
  return scr[kWarps];
}

// Sum of `n` doubles written by n CTAs (global, read through L2), returned to every thread.
__device__ __forceinline__ double sum_parts(const double* part, int n, double* scr) {
  double v = 0.0;
  for (int i = threadIdx.x; i < n; i += kThreads) v += ld_cg(part + i);
  return block_sum(v, scr);
}

// out_s[j] = sum_{b < nparts} part[b*stride + j], j < count.  Every CTA runs the same code on the
// same data, so all CTAs get bitwise identical results.  scr: kThreads doubles.
__device__ __forceinline__ void reduce_coef_parts(double* out_s, const double* part, int count, int nparts,
                                                  int stride, double* scr) {
  for (int j0 = 0; j0 < count; j0 += kThreads) {
    const int cnt = min(count - j0, kThreads);
    const int cp = (cnt + 31) & ~31;                 // lanes over j: coalesced 8-byte loads
    int nsub = kThreads / cp;
    if (nsub > nparts) nsub = nparts;
    const int sub = threadIdx.x / cp, j = threadIdx.x - sub * cp;
    double v = 0.0;
    if (sub < nsub && j < cnt) {
      const double* src = part + j0 + j;
#pragma unroll 4
      for (int b = sub; b < nparts; b += nsub) v += ld_cg(src + (size_t)b * stride);
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

// ------------------------------------------------------------------------------------ pass over the slab, transposed product
// For every column c:  x = src[rows, c];  (DEFL) x -= d[rows] * pdef[c];  (DST) dst[rows, c] = x;
//                      (DOT) part_out[c] = sum_rows x * t[rows]                       (S2 / S9 / A2)
//   gsrc, gdst   global matrices already offset to the CTA's first row; column stride ld
//   slab         shared-memory slab, column stride slab_ld (floats)
//   mb           rows this CTA owns;  N columns
//   t_s, d_s     shared: the CTA's rows of t and of the deflation vector;  pdef_s shared: N floats
//   part_out     global, N floats: this CTA's partial loads (written by lane lr == 0)
template <typename T, int VEC, int TR, int RC, int SRC, int DST, bool DEFL, bool DOT>
__device__ __forceinline__ void pass_t(const T* __restrict__ gsrc, T* __restrict__ gdst, long long ld,
                                       T* slab, int slab_ld, int mb, int N,
                                       const T* t_s, const T* d_s, const T* pdef_s,
                                       T* __restrict__ part_out) {
  constexpr int CW = 32 / TR;
  constexpr int CH = VEC * TR * RC;                    // rows per chunk
  constexpr int U = (RC >= 4) ? 2 : (RC == 2 ? 4 : 8);  // column groups in flight per warp
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int lr = lane % TR, lc = lane / TR;
  const int ngroups = (N + CW - 1) / CW;

  for (int r0 = 0; r0 < mb; r0 += CH) {
    T tv[RC][VEC], dv[RC][VEC];
    int roff[RC];
    bool rok[RC];
#pragma unroll
    for (int j = 0; j < RC; ++j) {
      roff[j] = r0 + (lr + TR * j) * VEC;
      rok[j] = roff[j] < mb;
#pragma unroll
      for (int e = 0; e < VEC; ++e) {
        tv[j][e] = (DOT && rok[j]) ? t_s[roff[j] + e] : T(0);
        dv[j][e] = (DEFL && rok[j]) ? d_s[roff[j] + e] : T(0);
      }
    }
    for (int g0 = w; g0 < ngroups; g0 += kWarps * U) {
      T x[U][RC][VEC];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int c = (g0 + u * kWarps) * CW + lc;
        const bool cok = c < N;
#pragma unroll
        for (int j = 0; j < RC; ++j) {
          if (cok && rok[j]) {
            if constexpr (SRC == SRC_GLOBAL) load_vec<T, VEC>(x[u][j], gsrc + (size_t)c * ld + roff[j]);
            else load_vec_smem<T, VEC>(x[u][j], slab + (size_t)c * slab_ld + roff[j]);
          } else {
#pragma unroll
            for (int e = 0; e < VEC; ++e) x[u][j][e] = T(0);
          }
        }
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int c = (g0 + u * kWarps) * CW + lc;
        const bool cok = c < N;
        T acc = T(0);
        const T pc = (DEFL && cok) ? pdef_s[c] : T(0);
#pragma unroll
        for (int j = 0; j < RC; ++j) {
          if constexpr (DEFL) {
#pragma unroll
            for (int e = 0; e < VEC; ++e) x[u][j][e] = fma_t(-dv[j][e], pc, x[u][j][e]);
          }
          if constexpr (DST != DST_NONE) {
            if (cok && rok[j]) {
              if constexpr (DST == DST_GLOBAL) store_vec<T, VEC>(gdst + (size_t)c * ld + roff[j], x[u][j]);
              else store_vec<T, VEC>(slab + (size_t)c * slab_ld + roff[j], x[u][j]);
            }
          }
          if constexpr (DOT) {
#pragma unroll
            for (int e = 0; e < VEC; ++e) acc = fma_t(x[u][j][e], tv[j][e], acc);
          }
        }
        if constexpr (DOT) {
#pragma unroll
          for (int o = 1; o < TR; o <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
          if (lr == 0 && cok) {
            if (r0 == 0) part_out[c] = acc;
            else part_out[c] = ld_cg(part_out + c) + acc;   // rare: more than one row chunk per CTA
          }
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------ pass over the slab, plain product
// t_out[rows] = sum_c src[rows, c] * p[c]                                             (S5)
// Columns are walked in DESCENDING order so that (streaming path) the columns the preceding
// ascending pass_t touched last are re-read while still in L2.
//   red_s  shared, kWarps * CH floats
template <typename T, int VEC, int TR, int RC, int SRC>
__device__ __forceinline__ void pass_n(const T* __restrict__ gsrc, long long ld, const T* slab, int slab_ld,
                                       int mb, int N, const T* p_s, T* t_out_s, T* red_s) {
  constexpr int CW = 32 / TR;
  constexpr int CH = VEC * TR * RC;
  constexpr int U = (RC >= 4) ? 2 : (RC == 2 ? 4 : 8);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int lr = lane % TR, lc = lane / TR;
  const int ngroups = (N + CW - 1) / CW;
  const int nsteps = (ngroups + kWarps * U - 1) / (kWarps * U);

  for (int r0 = 0; r0 < mb; r0 += CH) {
    int roff[RC];
    bool rok[RC];
    T acc[RC][VEC];
#pragma unroll
    for (int j = 0; j < RC; ++j) {
      roff[j] = r0 + (lr + TR * j) * VEC;
      rok[j] = roff[j] < mb;
#pragma unroll
      for (int e = 0; e < VEC; ++e) acc[j][e] = T(0);
    }
    for (int s = nsteps - 1; s >= 0; --s) {
      const int g0 = w + s * kWarps * U;
      T x[U][RC][VEC];
      T pc[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int c = (g0 + (U - 1 - u) * kWarps) * CW + lc;
        const bool cok = c < N;
        pc[u] = cok ? p_s[c] : T(0);
#pragma unroll
        for (int j = 0; j < RC; ++j) {
          if (cok && rok[j]) {
            if constexpr (SRC == SRC_GLOBAL) load_vec<T, VEC>(x[u][j], gsrc + (size_t)c * ld + roff[j]);
            else load_vec_smem<T, VEC>(x[u][j], slab + (size_t)c * slab_ld + roff[j]);
          } else {
#pragma unroll
            for (int e = 0; e < VEC; ++e) x[u][j][e] = T(0);
          }
        }
      }
#pragma unroll
      for (int u = 0; u < U; ++u)
#pragma unroll
        for (int j = 0; j < RC; ++j)
#pragma unroll
          for (int e = 0; e < VEC; ++e) acc[j][e] = fma_t(x[u][j][e], pc[u], acc[j][e]);
    }
    // combine the CW column groups of a warp, then the warps
#pragma unroll
    for (int j = 0; j < RC; ++j)
#pragma unroll
      for (int e = 0; e < VEC; ++e)
#pragma unroll
        for (int o = TR; o < 32; o <<= 1) acc[j][e] += __shfl_xor_sync(0xffffffffu, acc[j][e], o);
    __syncthreads();                                   // red_s free (previous chunk / caller)
    if (lc == 0) {
#pragma unroll
      for (int j = 0; j < RC; ++j)
#pragma unroll
        for (int e = 0; e < VEC; ++e) red_s[w * CH + (lr + TR * j) * VEC + e] = acc[j][e];
    }
    __syncthreads();
    for (int r = threadIdx.x; r < CH; r += kThreads) {
      if (r0 + r < mb) {
        T s = T(0);
#pragma unroll
        for (int q = 0; q < kWarps; ++q) s += red_s[q * CH + r];
        t_out_s[r0 + r] = s;
      }
    }
    __syncthreads();
  }
}

}  // namespace pca
