// =====================================================================================
// pca_reg.cuh -- register-resident single-sweep solve kernel (on-chip plan for matrices whose
// residual fits in the REGISTER FILES of the GPU: 4*M*N <= ~19 MB on 148 SMs; BASELINE.json
// configs 1, 2 and 5).
//
// Same iteration as pca_fused.cuh (rotated loop: the sweep that produces lambda' also produces
// the raw loads of the next pass; scores-side projection folded in by linearity through
// W = R^T V_(k); loads-side projection on the actual vector; PAPER.md:1016-1038 / :555-568), but
//   * the CTA's row block of R lives in REGISTERS for the whole solve (thread (g, gl) holds, for
//     each of the RPT rows of its row group g, the NV float4 column chunks 4*(gl + GT*v)): a sweep
//     t~ = R p, q = R^T t~ (S5 + S2) is 2*4*NV*RPT FMAs per thread plus one row reduction, with no
//     shared-memory or L2 traffic for R at all; the rank-1 deflation (S9) is applied in registers
//     the moment a component has converged;
//   * the CTA's rows of the unit score vectors V_(k) sit in shared memory (B-partials S6 and the
//     final t = t~ - V B never leave the SM);
//   * only Gs "slice owners" (a few CTAs) do the N-side work (combine the partial loads of their
//     column slice, W B and P A corrections, lambda', convergence test S8); the other CTAs go
//     straight from publishing their partials to waiting for the next p;
//   * for k > kdirect the k-vector B = V_(k)^T t~ is combined in two levels (every CTA sums a few
//     entries over all CTAs, the owners gather the k results) instead of every owner summing
//     all k entries over all CTAs;
//   * cross-CTA data travels in self-validating 8-byte words {payload, sequence number} that the
//     consumers poll directly (pca_fused.cuh, "LL exchange"); there is no grid barrier.
// =====================================================================================
#pragma once
#include "pca_fused.cuh"

namespace pca {

constexpr int kRegSmemRows = 2;   // RS of the compiled <GT, 2, 7, RS> variants: 2 of the 7 rows of a thread's row block in shared memory

struct RegParams {
  float* Rrm;            // M x ldr row-major residual (workspace): read once, written once
  float* T;              // M x K col-major
  float* P;              // N x K col-major
  float* lambda;         // K
  int* iters;            // K
  long long M;
  int N, K;
  double eps;
  int max_iter;
  int algo;              // 0 NIPALS, 1 GS
  int test_mode;         // 0 relative (listings), 1 absolute (text): pca_stagnated()
  int stag2;             // reading C4b: also compare lambda' with the value two passes back (PCA_OPT_STAGNATION)
  int out_svd;           // PCA_OPT_OUTPUT = 1: T holds the unit score vectors V (SVD triple V, U = P, Lambda)
  int defer_s3;          // PCA_OPT_DEFER_S3 (pca_fused.cuh, kDeferKappa)
  int G;                 // CTAs
  int Mb;                // rows per CTA (<= NG*RPT)
  int ldr;               // 4*NV*GT >= N
  int Ns, Gs;            // columns per slice owner (even), number of owners (CTAs 0..Gs-1); Gs*Ns == ldr
  int Kpad;              // K rounded up to 4
  int kdirect;           // B is combined in two levels for k > kdirect
  // LL exchange buffers (8-byte words {payload, seq}), double-buffered by the parity of the sweep number
  unsigned long long* Qx;   // [2][Gs][G][Ns]      partial raw loads, grouped by owner
  unsigned long long* SBx;  // [2][1 + Kpad/2][G][2] UNIT-major (a warp polling one unit over the parts reads contiguous
                            //                     words): unit 0 = partial |t~|^2 (fp64 bits), unit 1+j/2 = partial (B[j], B[j+1]) (fp32)
  unsigned long long* Bx;   // [2][2 + Kpad][2]    two-level: entry e as fp64 bits (entry 0 = |t~|^2, entry 2+j = B[j])
  unsigned long long* Ax;   // [2][Gs*Kpad]        partial A (fp32) of each owner; k <= 64: unit-major [Kpad/2][Gs][2] (a warp per unit,
                            //                     lanes over the owners), else owner-major [Gs][Kpad] (lanes over the units, owners in turn)
  unsigned long long* Px;   // [2][ldr]            p~ (loads before the loads-side projection, not normalised)
  unsigned long long* Nx;   // [2][Gs*2 + 6]       per owner: partial |p~|^2 (fp64, 2 words); then {decision, -, lambda' (fp64), rho (fp64)}
  unsigned long long* Pfx;  // [2][ldr]            final orthogonalised loads p^ of a component (buffer = component parity)
  unsigned long long* Nfx;  // [2][Gs*2]           per owner: partial |p^|^2 of the final loads
  unsigned* status;         // [0] != 0: an exchange wait gave up
  unsigned long long* trace;
  int trace_cap;
  // shared-memory carve-up (byte offsets)
  int off_p, off_ttil, off_d, off_qs, off_red, off_sgrp, off_B, off_A, off_scr, off_praw, off_vb, off_pc, off_wc;
  int off_x;             // >= 0 (one CTA only): the exchange buffers live in shared memory at this offset
  int off_rsm;           // kernel variants with RS > 0: the last RS rows of every row group live in shared memory (RowBlock)
};

// ------------------------------------------------------------------------------------ trace
// Phase trace (PCA_OPT_TRACE): thread 0 of EVERY CTA appends (phase << 56) | %globaltimer (ns, common to all SMs) to its
// slot (CTA b owns the records [b*cap/G, (b+1)*cap/G)), so that the timelines of the CTAs can be laid side by side.
// trace[0] = records written per slot (all CTAs write the same number).
__device__ __forceinline__ void reg_trace(const RegParams& prm, int& tn, int phase) {
  if (prm.trace_cap > 0 && threadIdx.x == 0) {
    const int capb = prm.trace_cap / prm.G;
    if (tn < capb) {
      extern __shared__ __align__(16) unsigned char trace_smem_[];
      const unsigned dep = *reinterpret_cast<volatile unsigned*>(trace_smem_);
      unsigned long long c;
      asm volatile("{ .reg .u32 t; and.b32 t, %1, 0; mov.u64 %0, %%globaltimer; }" : "=l"(c) : "r"(dep) : "memory");
      prm.trace[1 + (size_t)blockIdx.x * capb + tn] = ((unsigned long long)phase << 56) | (c & 0x00ffffffffffffffULL);
      ++tn;
    }
  }
}

// ------------------------------------------------------------------------------------ row reduction
// Eight values per lane, summed over the SEG lanes of a segment (SEG = 8, 16 or 32, a power of two).
// The first three butterfly steps halve the number of values instead of duplicating sums, so that
// 7 + (log2(SEG) - 3) shuffles do the work of 8*log2(SEG).  On return lane l holds the sum of
// value index  row = 4*bit(l, SEG/2) + 2*bit(l, SEG/4) + bit(l, SEG/8);  the SEG/8 lanes that
// differ only in the lower bits hold the same sum.
template <int SEG>
__device__ __forceinline__ float seg_reduce8(const float (&a)[8]) {
  const int lane = threadIdx.x & 31;
  const bool h1 = (lane & (SEG / 2)) != 0;
  float b[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const float keep = h1 ? a[4 + j] : a[j];
    const float send = h1 ? a[j] : a[4 + j];
    b[j] = keep + __shfl_xor_sync(0xffffffffu, send, SEG / 2);
  }
  const bool h2 = (lane & (SEG / 4)) != 0;
  float c[2];
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const float keep = h2 ? b[2 + j] : b[j];
    const float send = h2 ? b[j] : b[2 + j];
    c[j] = keep + __shfl_xor_sync(0xffffffffu, send, SEG / 4);
  }
  const bool h3 = (lane & (SEG / 8)) != 0;
  float d = (h3 ? c[1] : c[0]) + __shfl_xor_sync(0xffffffffu, h3 ? c[0] : c[1], SEG / 8);
#pragma unroll
  for (int o = SEG / 16; o > 0; o >>= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
  return d;
}

template <int SEG>
__device__ __forceinline__ int seg_row(int lane) {
  return (((lane & (SEG / 2)) != 0) ? 4 : 0) + (((lane & (SEG / 4)) != 0) ? 2 : 0) + (((lane & (SEG / 8)) != 0) ? 1 : 0);
}

template <int GT>
__device__ __forceinline__ void group_sync(int g) {
  if constexpr (GT <= 32) __syncwarp();
  else named_bar_sync(1 + g, GT);
}

// ------------------------------------------------------------------------------------ row block of a thread
// RPT rows x NV float4 of R per thread.  The first RPT - RS rows live in REGISTERS, the last RS in SHARED memory: the kernel is
// compiled for 128 registers per thread (512 threads, one CTA per SM) and 56 of them holding R (RPT = 7) left the rest of
// the pass spilling (428 bytes); shared memory is three quarters empty.  Every thread reads and writes only its own words
// there (no synchronisation), consecutive threads touch consecutive float4s (no bank conflicts).
template <int NV, int RPT, int RS>
struct RowBlock {
  static constexpr int RR = RPT - RS;
  float4 r[RR > 0 ? RR : 1][NV];
  float4* sm;      // this thread's float4 of the group's first shared-memory row
  int rstride;     // float4s between consecutive rows (ldr / 4)
  int vstride;     // float4s between the thread's column blocks (GT)
  __device__ __forceinline__ float4 get(int i, int v) const {
    if (i < RR) return r[i < RR ? i : 0][v];
    return sm[(i - RR) * rstride + v * vstride];
  }
  __device__ __forceinline__ void set(int i, int v, const float4& x) {
    if (i < RR) r[i < RR ? i : 0][v] = x;
    else sm[(i - RR) * rstride + v * vstride] = x;
  }
};

// ------------------------------------------------------------------------------------ sweeps
// FUSED sweep over the CTA's rows held in registers:
//   t~[r] = sum_n R[r,n] p[n]   (S5);   q[n] += R[r,n] t~[r]   (S2 of the next pass, :562,:1023)
// p_s holds the orthogonalised loads p^, pscale = 1/|p^|.
// Leaves t~ in ttil_s, the per-group partial q in qs[g][ldr], the per-group sum of t~^2 (fp64) in sgrp[g];
// ends with __syncthreads().  red_s: NG*WG*8 floats.
// WPRE (one-CTA kernel, GT < 32): the 32/GT row groups of a warp add their partial q by shuffles (fp32, fixed butterfly
// order) and the warp stores ONE row qs[warp][ldr] instead of one per group: a quarter / half of the rows to combine later.
template <int GT, int NV>
__device__ __forceinline__ void store_q_partial(float4 (&q4)[NV], float* qs, int g, int gl, int ldr, bool wpre) {
  if constexpr (GT < 32) {
    if (wpre) {
#pragma unroll
      for (int o = GT; o < 32; o <<= 1) {
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          q4[v].x += __shfl_xor_sync(0xffffffffu, q4[v].x, o);
          q4[v].y += __shfl_xor_sync(0xffffffffu, q4[v].y, o);
          q4[v].z += __shfl_xor_sync(0xffffffffu, q4[v].z, o);
          q4[v].w += __shfl_xor_sync(0xffffffffu, q4[v].w, o);
        }
      }
      if ((threadIdx.x & 31) < GT) {
#pragma unroll
        for (int v = 0; v < NV; ++v)
          *reinterpret_cast<float4*>(qs + (size_t)(threadIdx.x >> 5) * ldr + 4 * (gl + GT * v)) = q4[v];
      }
      return;
    }
  }
#pragma unroll
  for (int v = 0; v < NV; ++v) *reinterpret_cast<float4*>(qs + (size_t)g * ldr + 4 * (gl + GT * v)) = q4[v];
}

template <int GT, int NV, int RPT, bool WPRE = false, class RB>
__device__ __forceinline__ void reg_sweep_fused(const RB& Rr, const float* p_s, float pscale, float* ttil_s,
                                                float* qs, float* red_s, double* sgrp, int ldr) {
  static_assert(RPT <= 8, "one batch of at most 8 rows per group");
  constexpr int SEG = GT < 32 ? GT : 32;
  constexpr int WG = GT < 32 ? 1 : GT / 32;
  const int tid = threadIdx.x, g = tid / GT, gl = tid - g * GT, lane = tid & 31, wg = gl >> 5;
  float4 p4[NV], q4[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    p4[v] = *reinterpret_cast<const float4*>(p_s + 4 * (gl + GT * v));   // p = p^ / |p^| (S4)
    p4[v].x *= pscale; p4[v].y *= pscale; p4[v].z *= pscale; p4[v].w *= pscale;
    q4[v] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  float part[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    float a = 0.f;
    if (i < RPT) {
#pragma unroll
      for (int v = 0; v < NV; ++v) a = dot4(Rr.get(i < RPT ? i : 0, v), p4[v], a);
    }
    part[i] = a;
  }
  const float d = seg_reduce8<SEG>(part);
  float* rs = red_s + (size_t)g * (WG * 8);
  if ((lane & (SEG / 8 - 1)) == 0 || SEG == 8) rs[wg * 8 + seg_row<SEG>(lane)] = d;
  group_sync<GT>(g);
  float tt[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) tt[i] = 0.f;
#pragma unroll
  for (int w = 0; w < WG; ++w) {                                        // fixed order
    const float4 lo = *reinterpret_cast<const float4*>(rs + w * 8);
    const float4 hi = *reinterpret_cast<const float4*>(rs + w * 8 + 4);
    tt[0] += lo.x; tt[1] += lo.y; tt[2] += lo.z; tt[3] += lo.w;
    tt[4] += hi.x; tt[5] += hi.y; tt[6] += hi.z; tt[7] += hi.w;
  }
  if (gl == 0) {
    double sacc = 0.0;
#pragma unroll
    for (int i = 0; i < RPT; ++i) {
      ttil_s[g * RPT + i] = tt[i];
      sacc += (double)tt[i] * (double)tt[i];
    }
    sgrp[g] = sacc;
  }
#pragma unroll
  for (int i = 0; i < RPT; ++i)
#pragma unroll
    for (int v = 0; v < NV; ++v) axpy4(q4[v], Rr.get(i, v), tt[i]);
  store_q_partial<GT, NV>(q4, qs, g, gl, ldr, WPRE);
  __syncthreads();
}

// LOADS sweep at the start of component k:  t0 <- column k of the (already deflated) residual (S1,
// PAPER.md:556,:1017);  q = R^T t0 (S2).  Same outputs as reg_sweep_fused.
template <int GT, int NV, int RPT, bool WPRE = false, class RB>
__device__ __forceinline__ void reg_sweep_loads(const RB& Rr, int k, float* ttil_s, float* qs, double* sgrp,
                                                int ldr) {
  const int tid = threadIdx.x, g = tid / GT, gl = tid - g * GT;
  const int kc = k >> 2, ke = k & 3;
  if (gl == kc % GT) {
    const int kv = kc / GT;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      if (v == kv) {
#pragma unroll
        for (int i = 0; i < RPT; ++i) {
          const float4 x = Rr.get(i, v);
          ttil_s[g * RPT + i] = ke == 0 ? x.x : (ke == 1 ? x.y : (ke == 2 ? x.z : x.w));
        }
      }
    }
  }
  group_sync<GT>(g);
  float4 q4[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) q4[v] = make_float4(0.f, 0.f, 0.f, 0.f);
  double sacc = 0.0;
#pragma unroll
  for (int i = 0; i < RPT; ++i) {
    const float t = ttil_s[g * RPT + i];
    sacc += (double)t * (double)t;
#pragma unroll
    for (int v = 0; v < NV; ++v) axpy4(q4[v], Rr.get(i, v), t);
  }
  if (gl == 0) sgrp[g] = sacc;
  store_q_partial<GT, NV>(q4, qs, g, gl, ldr, WPRE);
  __syncthreads();
}

// ------------------------------------------------------------------------------------ LL reductions
// Sum over `nparts` parts of the 2-word unit at  base + part*stride + 2*u  (fp64, fixed order: lane l takes parts
// l, l+32, ... in order, then a shuffle tree).  PL = parts per lane kept in flight, UU = units in flight.
// If f64_unit0, unit 0 holds ONE fp64 value in its two words.  The sums are returned in every lane.
template <int PL>
__device__ __forceinline__ void reg_ll_unit(const u64* base, int stride, int nparts, int u, bool f64, unsigned seq,
                                            unsigned* status, double& r0, double& r1) {
  const int lane = threadIdx.x & 31;
  double a0 = 0.0, a1 = 0.0;
  for (int b0 = lane; b0 < nparts; b0 += 32 * PL) {
    u64 x[PL], y[PL];
#pragma unroll
    for (int i = 0; i < PL; ++i) {
      const int bq = b0 + 32 * i;
      x[i] = 0; y[i] = 0;
      if (bq < nparts) gl_ld2(base + (size_t)bq * stride + 2 * u, x[i], y[i]);
    }
#pragma unroll
    for (int i = 0; i < PL; ++i) {
      const int bq = b0 + 32 * i;
      if (bq < nparts) {
        gl_wait2(base + (size_t)bq * stride + 2 * u, seq, x[i], y[i], status);
        if (f64) a0 += ll_d(x[i], y[i]);
        else { a0 += (double)ll_f(x[i]); a1 += (double)ll_f(y[i]); }
      }
    }
  }
  r0 = warp_sum(a0);
  r1 = warp_sum(a1);
}

// Few parts (nparts <= 32): four units in flight per warp.
__device__ __forceinline__ void reg_ll_units4(const u64* base, int stride, int ustride, int nparts, int u0, int ustep, int units,
                                              unsigned seq, unsigned* status, double* out) {
  const int lane = threadIdx.x & 31;
  u64 x[4], y[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int u = u0 + i * ustep;
    x[i] = 0; y[i] = 0;
    if (u < units && lane < nparts) gl_ld2(base + (size_t)lane * stride + (size_t)u * ustride, x[i], y[i]);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int u = u0 + i * ustep;
    if (u < units) {                                                    // warp-uniform
      double a0 = 0.0, a1 = 0.0;
      if (lane < nparts) {
        gl_wait2(base + (size_t)lane * stride + (size_t)u * ustride, seq, x[i], y[i], status);
        a0 = (double)ll_f(x[i]); a1 = (double)ll_f(y[i]);
      }
      a0 = warp_sum(a0);
      a1 = warp_sum(a1);
      if (lane == 0) { out[2 * u] = a0; out[2 * u + 1] = a1; }
    }
  }
}

// out[2u], out[2u+1] for all units u < units (fp32 payloads), every warp of the CTA taking part.  No barrier inside.
__device__ __forceinline__ void reg_ll_reduce_all(const u64* base, int stride, int ustride, int nparts, int units, unsigned seq,
                                                  unsigned* status, double* out) {
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (nparts <= 32) {
    for (int u0 = w; u0 < units; u0 += 4 * kWarps) reg_ll_units4(base, stride, ustride, nparts, u0, kWarps, units, seq, status, out);
  } else {
    for (int u = w; u < units; u += kWarps) {
      double a0, a1;
      reg_ll_unit<5>(base + (size_t)u * ustride, stride, nparts, 0, false, seq, status, a0, a1);
      if (lane == 0) { out[2 * u] = a0; out[2 * u + 1] = a1; }
    }
  }
}

// Combine the NG group partials of a sweep (fixed order) and publish this CTA's partial raw loads:
// column c of slice owner o = c / Ns goes to Qpar[(o*G + b)*Ns + c % Ns]   (S2)
template <int GT>
__device__ __forceinline__ void reg_publish_q(const RegParams& prm, const float* qs, u64* Qpar, int b, unsigned seq) {
  constexpr int NG = kThreads / GT;
  const int ldr = prm.ldr, Ns = prm.Ns;
  for (int c = threadIdx.x * 2; c < ldr; c += kThreads * 2) {
    float2 a = *reinterpret_cast<const float2*>(qs + c);
#pragma unroll 8
    for (int g = 1; g < NG; ++g) {
      const float2 v = *reinterpret_cast<const float2*>(qs + (size_t)g * ldr + c);
      a.x += v.x; a.y += v.y;
    }
    const int o = c / Ns, i = c - o * Ns;
    gl_st2(Qpar + ((size_t)o * prm.G + b) * Ns + i, ll_wordf(a.x, seq), ll_wordf(a.y, seq));
  }
}

// Publish |t~|^2 and (GS-PCA, k > 0) the B-partials V_b^T t~ (S6) of this CTA.
// Vb: [rows][KV] unit score rows of this CTA (shared memory, odd row stride KV: conflict-free for lanes over rows AND
// over columns).  `parts` threads (consecutive lanes) share a column j and split the rows; no barrier inside.
// B-partials of reg_publish_sb with a compile-time number of lanes per column (PARTS): shifts and an unrolled shuffle tree
template <int PARTS>
__device__ __forceinline__ void reg_publish_b_t(const float* Vb, int KV, const float* ttil_s, u64* sbx, int G, int mb, int k,
                                                unsigned seq) {
  constexpr int parts = PARTS;
  const int tid = threadIdx.x;
  const int j = tid / parts, part = tid - j * parts;
  float a = 0.f;
  if (j < k)
  {
    float a1 = 0.f, a2 = 0.f, a3 = 0.f;                                  // four independent chains (fixed association)
    int r = part;
    for (; r + 3 * parts < mb; r += 4 * parts) {                       // (no trip when a thread has fewer than 4 rows)
      a = fmaf(Vb[(size_t)r * KV + j], ttil_s[r], a);
      a1 = fmaf(Vb[(size_t)(r + parts) * KV + j], ttil_s[r + parts], a1);
      a2 = fmaf(Vb[(size_t)(r + 2 * parts) * KV + j], ttil_s[r + 2 * parts], a2);
      a3 = fmaf(Vb[(size_t)(r + 3 * parts) * KV + j], ttil_s[r + 3 * parts], a3);
    }
    for (; r < mb; r += parts) a = fmaf(Vb[(size_t)r * KV + j], ttil_s[r], a);
    a = (a + a1) + (a2 + a3);
  }
#pragma unroll
  for (int o = parts >> 1; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  const float nb = __shfl_down_sync(0xffffffffu, a, parts);             // column j + 1 (same part)
  if (part == 0 && (j & 1) == 0 && j < k)
    gl_st2(sbx + (size_t)(1 + (j >> 1)) * G * 2, ll_wordf(a, seq), ll_wordf(j + 1 < k ? nb : 0.f, seq));
}
__device__ __forceinline__ void reg_publish_sb(const float* Vb, int KV, const float* ttil_s, const double* sgrp, u64* sbx, int G,
                                               int NG, int mb, int k, bool with_b, unsigned seq) {   // sbx: this CTA's slot of unit 0
  const int tid = threadIdx.x;
  if (tid == 0) {
    double a = 0.0;
    for (int g = 0; g < NG; ++g) a += sgrp[g];
    gl_st2d(sbx, a, seq);
  }
  if (!with_b) return;
  __syncwarp();            // (warp 0 re-converges before the full-mask shuffles below; measured in pca_fused.cuh: 2-6 x otherwise)
  int Kc = 32;
  while (Kc < k) Kc <<= 1;
  switch (kThreads / Kc) {                                             // lanes per column: 1..16, a power of two
    case 16: reg_publish_b_t<16>(Vb, KV, ttil_s, sbx, G, mb, k, seq); break;
    case 8: reg_publish_b_t<8>(Vb, KV, ttil_s, sbx, G, mb, k, seq); break;
    case 4: reg_publish_b_t<4>(Vb, KV, ttil_s, sbx, G, mb, k, seq); break;
    case 2: reg_publish_b_t<2>(Vb, KV, ttil_s, sbx, G, mb, k, seq); break;
    default: reg_publish_b_t<1>(Vb, KV, ttil_s, sbx, G, mb, k, seq); break;
  }
}


// praw[i] -= sum_{j<k} C[i*KP + j] * coef[j] for the ns columns of this owner: LPR lanes per column (8 for k <= 64, else 32;
// lane l takes j = l, l + LPR, ... in order, then a shuffle tree), 32/LPR columns per warp and round.
template <int LPR>
__device__ __forceinline__ void reg_slice_correct_t(double* praw_s, const float* C, int KP, const double* coef_s, int ns, int k) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  constexpr int rpw = 32 / LPR;
  const int ll = lane & (LPR - 1);
  for (int i0 = 0; i0 < ns; i0 += rpw * kWarps) {                             // (uniform trip count: shuffles inside)
    const int i = i0 + w * rpw + lane / LPR;
    double c = 0.0;
    if (i < ns) {
      const float* ci = C + (size_t)i * KP;
#pragma unroll 4
      for (int j = ll; j < k; j += LPR) c += (double)ci[j] * coef_s[j];
    }
#pragma unroll
    for (int o = LPR >> 1; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (ll == 0 && i < ns) praw_s[i] -= c;
  }
}
__device__ __forceinline__ void reg_slice_correct(double* praw_s, const float* C, int KP, const double* coef_s, int ns, int k) {
  if (k <= 64) reg_slice_correct_t<8>(praw_s, C, KP, coef_s, ns, k);          // (compile-time lane count: unrolled shuffle tree)
  else reg_slice_correct_t<32>(praw_s, C, KP, coef_s, ns, k);
}

// S3, first half: this owner's partial  a_S[j] = sum_{n in S} P[n,j] p~[n], all threads of the CTA.
__device__ __forceinline__ void reg_publish_a(const float* Pc, int KP, const double* praw_s, u64* ax, int ustride, int ns, int k,
                                              unsigned seq) {   // ax: this owner's slot of unit 0; ustride: words between units
  const int tid = threadIdx.x;
  int Kc = 32;
  while (Kc < k) Kc <<= 1;
  const int parts = kThreads / Kc;
  const int j = tid / parts, part = tid - j * parts;
  double a = 0.0;
  if (j < k)
    for (int i = part; i < ns; i += parts) a += (double)Pc[(size_t)i * KP + j] * praw_s[i];
  for (int o = parts >> 1; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  const double nb = __shfl_down_sync(0xffffffffu, a, parts);
  if (part == 0 && (j & 1) == 0 && j < k)
    gl_st2(ax + (size_t)(j >> 1) * ustride, ll_wordf((float)a, seq), ll_wordf(j + 1 < k ? (float)nb : 0.f, seq));
}

// A = sum over the owners of their partials, published with tag `tag` in parity buffer `par`; all threads
// of the CTA; the caller synchronises before reading A_s.  scratch: kThreads double2 (k > 64 only).
__device__ __forceinline__ void reg_gather_a(const RegParams& prm, const u64* Ax, unsigned par, unsigned tag, int k, float* scratch,
                                             double* A_s, unsigned* status) {
  const int Gs = prm.Gs, Kpad = prm.Kpad;
  if (k <= 64) {                                                      // few units: a warp per unit, lanes over the owners
    reg_ll_reduce_all(Ax + (size_t)par * Gs * Kpad, 2, Gs * 2, Gs, (k + 1) >> 1, tag, status, A_s);
  } else {                                                            // many units: lanes over the units (coalesced), owners in turn
    RegGather ga;
    const int ua = (k + 1) >> 1;
    int ha = 1;
    while (ha < ua) ha <<= 1;
    ga.base = Ax + (size_t)par * Gs * Kpad; ga.stride = Kpad; ga.hp = ha; ga.npairs = ua; ga.nparts = Gs;
    ga.f64_pair0 = 0; ga.red = reinterpret_cast<double2*>(scratch); ga.out = A_s;
    u64 ax8[8], ay8[8];
    reg_gather_issue<8>(ga, ax8, ay8);
    reg_gather_finish<8>(ga, ax8, ay8, tag, status);
    __syncthreads();
    reg_gather_store(ga);
  }
}

// ------------------------------------------------------------------------------------ the kernel
template <int GT, int NV, int RPT, int RS = 0>          // RS: rows of the thread's row block kept in shared memory (RowBlock)
__global__ void __launch_bounds__(kThreads, 1) pca_reg_kernel(const RegParams prm) {
  extern __shared__ __align__(16) unsigned char smem[];
  constexpr int NG = kThreads / GT;
  float* p_s = reinterpret_cast<float*>(smem + prm.off_p);        // 2 x ldr: orthogonalised loads p^, double-buffered by the pass
                                                                  // parity (the gather that reports "done" carries no loads)
  float* ttil_s = reinterpret_cast<float*>(smem + prm.off_ttil);  // NG*RPT: t0 / t~ rows of this CTA
  float* d_s = reinterpret_cast<float*>(smem + prm.off_d);        // NG*RPT: deflation vector rows
  float* qs = reinterpret_cast<float*>(smem + prm.off_qs);        // NG x ldr group partials
  float* red_s = reinterpret_cast<float*>(smem + prm.off_red);    // kThreads: row-reduction scratch
  double* sgrp = reinterpret_cast<double*>(smem + prm.off_sgrp);  // NG
  double* sb_s = reinterpret_cast<double*>(smem + prm.off_B);     // 4 + Kpad: |t~|^2, -, B
  double* B_s = sb_s + 2;
  double* A_s = reinterpret_cast<double*>(smem + prm.off_A);      // Kpad + 2
  double* scr = reinterpret_cast<double*>(smem + prm.off_scr);    // kThreads
  double* ctl_s = scr + kThreads - 8;                             // [0] lambda' [1] decision (owners' test); [2] 1/|p^| [3] lambda' [4] decision (gathered)
  double* praw_s = reinterpret_cast<double*>(smem + prm.off_praw);// Ns: p~ / p^ slice of this owner
  float* Vb = reinterpret_cast<float*>(smem + prm.off_vb);        // NG*RPT x Kpad: unit score rows of this CTA
  float* Pc = reinterpret_cast<float*>(smem + prm.off_pc);        // Ns x Kpad: P[slice, :]   (owners)
  float* Wc = reinterpret_cast<float*>(smem + prm.off_wc);        // Ns x Kpad: W[slice, :] = (R^T V)[slice, :]

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int g = tid / GT, gl = tid - g * GT;
  const int b = blockIdx.x;
  const long long M = prm.M;
  const int N = prm.N, K = prm.K, G = prm.G, ldr = prm.ldr, Kpad = prm.Kpad, Ns = prm.Ns, Gs = prm.Gs;
  u64 *Qx = prm.Qx, *SBx = prm.SBx, *Bx = prm.Bx, *Ax = prm.Ax, *Px = prm.Px, *Nx = prm.Nx, *Pfx = prm.Pfx, *Nfx = prm.Nfx;
  const int NXW = Gs * 2 + 6;                                      // words per parity buffer of Nx
  if (prm.off_x >= 0) {                                            // one CTA: exchange through shared memory
    u64* xb = reinterpret_cast<u64*>(smem + prm.off_x);
    Qx = xb; SBx = Qx + 2 * (size_t)ldr; Bx = SBx + 4 * (1 + (Kpad >> 1)); Ax = Bx + 4 * (2 + Kpad); Px = Ax + 4 * (Kpad >> 1);
    Nx = Px + 2 * (size_t)ldr; Pfx = Nx + 2 * NXW; Nfx = Pfx + 2 * (size_t)ldr;
    const int nw = (int)(Nfx + 2 * (Gs * 2) - xb);
    for (int i = tid; i < nw; i += kThreads) xb[i] = 0ULL;         // sequence numbers start at 0
  }
  double* pt_s = praw_s + Ns;                                      // Ns: R^T t slice (p~ before the loads-side projection), for W
  const int UB = 1 + (Kpad >> 1);                                  // 2-word units per parity buffer of SBx
  const int KV = Kpad | 1;                                         // odd row stride of the shared-memory panels Vb, Pc, Wc
  const bool gs = prm.algo == 1;
  const long long m0 = (long long)b * prm.Mb;
  const int mb = (int)max(0LL, min((long long)prm.Mb, M - m0));
  const bool owner = b < Gs;
  const int n0 = b * Ns;
  const int ns = owner ? max(0, min(Ns, N - n0)) : 0;
  unsigned seq = 0;
  unsigned* status = prm.status;
  int tn = 0;
  double bf2 = 0.0;                                                // sum over the finished components of |B_j|^2 (kDeferKappa)
  float* Rb = prm.Rrm + (size_t)m0 * ldr;
  float* Tb = prm.T + m0;

  // ---- R <- X: this thread's part of the CTA's row block, into registers ----
  RowBlock<NV, RPT, RS> Rr;
  Rr.sm = reinterpret_cast<float4*>(smem + prm.off_rsm) + (size_t)(g * RS) * (ldr >> 2) + gl;
  Rr.rstride = ldr >> 2;
  Rr.vstride = GT;
#pragma unroll
  for (int i = 0; i < RPT; ++i) {
    const int r = g * RPT + i;
#pragma unroll
    for (int v = 0; v < NV; ++v)
      Rr.set(i, v, (r < mb) ? ld_stream4(Rb + (size_t)r * ldr + 4 * (gl + GT * v)) : make_float4(0.f, 0.f, 0.f, 0.f));
  }
  for (int i = tid; i < NG * RPT; i += kThreads) { d_s[i] = 0.f; ttil_s[i] = 0.f; }
  for (int n = tid; n < 2 * ldr; n += kThreads) p_s[n] = 0.f;
  for (int i = tid; i < Ns; i += kThreads) praw_s[i] = 0.0;
  __syncthreads();

  for (int k = 0; k < K; ++k) {
    const bool gsk = gs && k > 0;
    const bool two = gsk && k > prm.kdirect;
    const int U = 1 + ((k + 1) >> 1);                              // 2-word units of [ |t~|^2 | B ]
    reg_trace(prm, tn, TR_COMPONENT);
    // ---- S1 + S2: t0 <- column k of the deflated residual; q = R^T t0 ----
    reg_sweep_loads<GT, NV, RPT>(Rr, k, ttil_s, qs, sgrp, ldr);
    ++seq;
    {
      const unsigned par = seq & 1u;
      reg_publish_q<GT>(prm, qs, Qx + (size_t)par * Gs * G * Ns, b, seq);
      reg_publish_sb(Vb, KV, ttil_s, sgrp, SBx + ((size_t)par * UB * G + b) * 2, G, NG, mb, k, false, seq);
    }
    reg_trace(prm, tn, TR_LOADS_DONE);

    double lam = 0.0, lam2 = 0.0, lam_new = 0.0;                    // lambda of the previous pass, of the one before, of this one
    float rhof = 1.f;                                               // |p~|/|p^| of the pass that converged (S3, deferred)
    bool deferred = false;                                          // the loads of the pass in flight are p~, not p^
    int it = 0;
    bool degenerate = false, first = true;
    float pscale = 0.f;
    for (;;) {
      const unsigned par = seq & 1u;
      const bool with_b = gsk && !first;
      const bool two_now = with_b && two;
      // ---- hop 1: owners combine their slice of the raw loads; |t~|^2 and B either directly (owners) or in two levels ----
      if (two_now) {
        // level 1: the 2-word units of [ |t~|^2 | B ] are dealt out to the duty CTAs (the non-owners if there are enough)
        const int duty0 = (G - Gs >= 16) ? Gs : 0, nduty = G - duty0;
        if (b >= duty0) {
          const u64* sbase = SBx + (size_t)par * UB * G * 2;
          for (int u = (b - duty0) + w * nduty; u < U; u += kWarps * nduty) {
            double a0, a1;
            reg_ll_unit<5>(sbase + (size_t)u * G * 2, 2, G, 0, u == 0, seq, status, a0, a1);
            if (lane == 0) {
              u64* bx = Bx + ((size_t)par * (2 + Kpad) + 2 * u) * 2;
              gl_st2d(bx, a0, seq);
              gl_st2d(bx + 2, a1, seq);
            }
          }
        }
      }
      if (owner) {
        RegGather gq;
        gq.base = Qx + ((size_t)par * Gs + b) * G * Ns; gq.stride = Ns; gq.hp = min(Ns >> 1, kThreads); gq.npairs = Ns >> 1;
        gq.nparts = G; gq.f64_pair0 = false; gq.red = reinterpret_cast<double2*>(qs); gq.out = praw_s;
        // [ |t~|^2 | B ] summed directly: warp u takes unit u (<= 16 units, plan: kdirect <= 30), lanes over the parts (contiguous)
        const int usb = two_now ? 0 : (1 + (with_b ? ((k + 1) >> 1) : 0));
        const u64* ub = SBx + ((size_t)par * UB + w) * G * 2;
        u64 sx[5], sy[5];
        const bool sbw = w < usb && (w > 0 || b == 0);                       // |t~|^2 (unit 0) is read by owner 0 only: it alone tests
        if (sbw) {
#pragma unroll
          for (int i2 = 0; i2 < 5; ++i2) {
            const int part = lane + 32 * i2;
            sx[i2] = 0; sy[i2] = 0;
            if (part < G) gl_ld2(ub + (size_t)part * 2, sx[i2], sy[i2]);
          }
        }
        __syncthreads();                                                      // qs (group partials of the sweep) is free
        if (with_b) {
          // deferred loads-side Gram-Schmidt (see "S3, deferred" below): every owner sums the A-partials the owners published
          // one pass ago (they have been there for a whole sweep): |p^|^2 = |p~|^2 - |A|^2 for owner 0's test, and the
          // decision whether the next pass may defer again
          reg_gather_a(prm, Ax, (seq - 1u) & 1u, seq - 1u, k, qs, A_s, status);
          __syncthreads();
          if (w == 0) {
            double a2 = 0.0;
            for (int j = lane; j < k; j += 32) a2 += A_s[j] * A_s[j];
            a2 = warp_sum(a2);
            if (lane == 0) ctl_s[6] = a2;
          }
        }
        if ((Ns >> 1) <= kThreads) {
          u64 qx[5], qy[5];
          reg_gather_issue<5>(gq, qx, qy);
          reg_gather_finish<5>(gq, qx, qy, seq, status);
        } else {                                                              // very wide slices (few CTAs): a pair per thread
          for (int pr2 = tid; pr2 < (Ns >> 1); pr2 += kThreads) {
            double a0 = 0.0, a1 = 0.0;
            for (int part = 0; part < G; ++part) {
              u64 xx = 0, yy = 0;
              gl_wait2(gq.base + (size_t)part * Ns + 2 * pr2, seq, xx, yy, status);
              a0 += (double)ll_f(xx); a1 += (double)ll_f(yy);
            }
            praw_s[2 * pr2] = a0; praw_s[2 * pr2 + 1] = a1;
          }
        }
        if (sbw) {
          double a0 = 0.0, a1 = 0.0;
#pragma unroll
          for (int i2 = 0; i2 < 5; ++i2) {
            const int part = lane + 32 * i2;
            if (part < G) {
              gl_wait2(ub + (size_t)part * 2, seq, sx[i2], sy[i2], status);
              if (w == 0) a0 += ll_d(sx[i2], sy[i2]);
              else { a0 += (double)ll_f(sx[i2]); a1 += (double)ll_f(sy[i2]); }
            }
          }
          for (int part = lane + 160; part < G; part += 32) {
            u64 xx = 0, yy = 0;
            gl_wait2(ub + (size_t)part * 2, seq, xx, yy, status);
            if (w == 0) a0 += ll_d(xx, yy);
            else { a0 += (double)ll_f(xx); a1 += (double)ll_f(yy); }
          }
          a0 = warp_sum(a0);
          a1 = warp_sum(a1);
          if (lane == 0) { sb_s[2 * w] = a0; sb_s[2 * w + 1] = a1; }
        }
        if ((Ns >> 1) <= kThreads) {
          __syncthreads();
          reg_gather_store(gq);
        }
        if (two_now) {                                                        // hop 1b: gather |t~|^2 and B
          const u64* bx = Bx + (size_t)par * (2 + Kpad) * 2;
          for (int e = tid; e < 2 * U; e += kThreads) {
            u64 x = 0, y = 0;
            gl_wait2(bx + 2 * e, seq, x, y, status);
            sb_s[e] = ll_d(x, y);
          }
        }
        __syncthreads();
        reg_trace(prm, tn, TR_X1);
        // S7/S8 by warp 0 of owner 0 (then it joins the others);  p~ = q - W B on the owner's slice (needs only B)
        // (the LAST warp: the slice correction below starts with warp 0 and reaches the last warp only for slices wider than
        //  60 columns, so on owner 0 the scalar chain of the test runs beside it instead of in front of it)
        if (w == kWarps - 1 && lane == 0 && (b != 0 || first)) ctl_s[7] = 1.0;
        if (w == kWarps - 1 && b != 0 && lane == 0) { ctl_s[0] = 0.0; reinterpret_cast<int*>(ctl_s + 1)[0] = 0; }
        if (w == kWarps - 1 && b == 0) {
          const double s = sb_s[0];
          int st = 0;                                                         // 0 continue, 1 done, 2 degenerate
          double ln = 0.0;
          if (first) {
            if (!(s > 0.0)) st = 2;                                           // zero start column (C7)
          } else {
            double bb = 0.0;
            if (gsk) {                                                        // B = V_(k)^T t~
              for (int j = lane; j < k; j += 32) bb += B_s[j] * B_s[j];
              bb = warp_sum(bb);
            }
            double l2 = s - bb;                                               // |t~ - V B|^2, V orthonormal
            double rho = 1.0, rho2 = 1.0;
            if (gsk && deferred) {                                            // |p^|^2 = |p~|^2 - |A|^2 (P orthonormal)
              const double pn2 = ctl_s[5], d2 = pn2 - ctl_s[6];
              if (!(d2 > 0.0)) l2 = 0.0;
              else rho2 = pn2 * fast_rcp(d2);
              l2 *= rho2;
              rho = fast_sqrt(rho2);
            }
            if (lane == 0) ctl_s[7] = rho;
            if (!(l2 > 0.0)) st = 2;                                          // reading C7
            else {
              ln = fast_sqrt(l2);                                                  // S7
              // S8: the listings' strict relative test (reading C3)
              // (+ reading C4b: in fp32 the iteration can end in a period-2 limit cycle, lambda' alternating between two
              //  values; that is stagnation too, so lambda' is also compared with the value two passes back)
              if (pca_stagnated(lam, lam2, ln, prm.eps, prm.test_mode, prm.stag2) || (it >= prm.max_iter)) st = 1;
            }
          }
          if (lane == 0) { ctl_s[0] = ln; reinterpret_cast<int*>(ctl_s + 1)[0] = st; }
        }
        __syncwarp();
        if (with_b) reg_slice_correct(praw_s, Wc, KV, B_s, ns, k);
        __syncthreads();
        // S3: a_S[j] = sum_{n in S} P[n,j] p~[n]
        if (gs)
          for (int i2 = tid; i2 < Ns; i2 += kThreads) pt_s[i2] = praw_s[i2];
        const int st = reinterpret_cast<const int*>(ctl_s + 1)[0];
        reg_trace(prm, tn, TR_TEST);
        // ---- S3, deferred.  The paper orthogonalises the loads first, p^ = p~ - P_(k) A, and multiplies then,
        // t~ = R p^.  R P_(k) lies in span V_(k) (deflation: R_(j+1) p_j = t~_j - t_j = V_(j) B_j, later deflations add multiples
        // of v_i), and the scores-side projection t = t~ - V_(k) V_(k)^T t~ removes that span, so R p~ and R p^
        // give the SAME t: the sweep starts from p~ without waiting for A = sum of the owners' partials (one dependent cross-CTA
        // hop less per pass).  The iteration needs |p^|^2 = |p~|^2 - |A|^2 (owner 0, at the next test); p^ itself is formed once,
        // when the component has converged ("final loads" below).  (The two-sweep kernel keeps the paper's literal order.)
        // Deferring costs accuracy when A is NOT small (the first pass of a component starts from a raw column; fixed-pass runs
        // never converge): t~ then carries a large component in span V_(k) and lambda'^2 = |t~|^2 - |B|^2 cancels.  So the first
        // two passes of a component, and every pass for which the bound of kDeferKappa (pca_fused.cuh) fails, take the paper's
        // order (hop 2).  Every owner takes the same decision from the same numbers.
        const bool defer_now = prm.defer_s3 != 0 && with_b && ctl_s[6] * bf2 <= kDeferKappa * ctl_s[5] * lam * lam;
        if (gsk && !defer_now) {
          if (k <= 64) reg_publish_a(Pc, KV, praw_s, Ax + (size_t)par * Gs * Kpad + (size_t)b * 2, Gs * 2, ns, k, seq);
          else reg_publish_a(Pc, KV, praw_s, Ax + ((size_t)par * Gs + b) * Kpad, 2, ns, k, seq);
          // ---- hop 2: A = sum of the owners' partials;  p^ = p~ - P_(k) A ----
          reg_gather_a(prm, Ax, par, seq, k, qs, A_s, status);
          __syncthreads();
          reg_trace(prm, tn, TR_X2);
          reg_slice_correct(praw_s, Pc, KV, A_s, ns, k);
          __syncthreads();
        }
        // ---- publish the p~ slice, its squared norm, the decision, lambda' and rho ----
        if (w == 0) {
          double q2 = 0.0;
          for (int u = lane; 2 * u < Ns; u += 32) {
            const float v0 = (2 * u < ns) ? (float)praw_s[2 * u] : 0.f;
            const float v1 = (2 * u + 1 < ns) ? (float)praw_s[2 * u + 1] : 0.f;
            gl_st2(Px + (size_t)par * ldr + n0 + 2 * u, ll_wordf(v0, seq), ll_wordf(v1, seq));
            q2 += (double)v0 * (double)v0 + (double)v1 * (double)v1;
          }
          q2 = warp_sum(q2);
          if (lane == 0) {
            u64* nx = Nx + (size_t)par * NXW;
            gl_st2d(nx + (size_t)b * 2, q2, seq);
            if (b == 0) {                                                     // every owner takes the same decision: owner 0 reports it
              gl_st2(nx + (size_t)Gs * 2, ll_word((unsigned)st, seq), ll_word(defer_now ? 1u : 0u, seq));
              gl_st2d(nx + (size_t)Gs * 2 + 2, ctl_s[0], seq);
              if (gsk) gl_st2d(nx + (size_t)Gs * 2 + 4, ctl_s[7], seq);
            }
          }
          __syncwarp();
        }
        reg_trace(prm, tn, TR_PHAT);
        // S3, first half, off the critical path: a_S[j] = sum_{n in S} P[n,j] p~[n]
        if (gsk && defer_now) {
          if (k <= 64) reg_publish_a(Pc, KV, praw_s, Ax + (size_t)par * Gs * Kpad + (size_t)b * 2, Gs * 2, ns, k, seq);
          else reg_publish_a(Pc, KV, praw_s, Ax + ((size_t)par * Gs + b) * Kpad, 2, ns, k, seq);
        }
      }
      // ---- arrival hint: ONE thread of the CTA polls ONE word (the last owner's norm record) while the others sleep at the
      // barrier; only then does every thread load its words of p^ (each validated by its own sequence number, so the hint
      // orders nothing).  Measured: with all 148 x 512 threads polling the same 8 KB the hop takes 2.9-3.3 us, this way 1.8 us.
      if (tid == (kWarps - 1) * 32) {
        const u64* nxl = Nx + (size_t)par * NXW + (size_t)(Gs - 1) * 2;
        u64 x = 0, y = 0;
        gl_wait2(nxl, seq, x, y, status);
      }
      __syncthreads();
      // ---- hop 3 (every CTA): gather p^, |p^|^2, the decision and lambda' ----
      if (w == kWarps - 1) {
        const u64* nx = Nx + (size_t)par * NXW;
        double nsum = 0.0, lamv = 0.0;
        unsigned stv = 0;
        u64 x1 = 0, y1 = 0, x2 = 0, y2 = 0, x3 = 0, y3 = 0;
        double rhov = 1.0;
        if (lane == 0) { gl_ld2(nx + (size_t)Gs * 2, x1, y1); gl_ld2(nx + (size_t)Gs * 2 + 2, x2, y2); if (gsk) gl_ld2(nx + (size_t)Gs * 2 + 4, x3, y3); }
        for (int o = lane; o < Gs; o += 32) {
          u64 x0 = 0, y0 = 0;
          gl_wait2(nx + (size_t)o * 2, seq, x0, y0, status);
          nsum += ll_d(x0, y0);
        }
        if (lane == 0) {
          gl_wait2(nx + (size_t)Gs * 2, seq, x1, y1, status);
          gl_wait2(nx + (size_t)Gs * 2 + 2, seq, x2, y2, status);
          if (gsk) gl_wait2(nx + (size_t)Gs * 2 + 4, seq, x3, y3, status);
          stv = (unsigned)x1;
          reinterpret_cast<int*>(ctl_s + 1)[1] = (int)(unsigned)y1;             // the loads just published are p~ (S3 deferred)
          lamv = ll_d(x2, y2);
          if (gsk) rhov = ll_d(x3, y3);
        }
        nsum = warp_sum(nsum);
        if (lane == 0) {
          reinterpret_cast<float*>(ctl_s + 2)[0] = (nsum > 0.0) ? (float)rsqrt(nsum) : 0.f;
          ctl_s[3] = lamv;
          reinterpret_cast<int*>(ctl_s + 4)[0] = (int)stv;
          reinterpret_cast<float*>(ctl_s + 4)[1] = (float)rhov;
          ctl_s[5] = nsum;                                                    // |p~|^2 of the loads the next sweep runs with
        }
      }
      {
        const u64* px = Px + (size_t)par * ldr;
        float* pg = p_s + (size_t)(it & 1) * ldr;
        for (int u0 = tid; 2 * u0 < ldr; u0 += kThreads * 4) {
          u64 x[4], y[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int u = u0 + i * kThreads;
            x[i] = 0; y[i] = 0;
            if (2 * u < ldr) gl_ld2(px + 2 * u, x[i], y[i]);
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int u = u0 + i * kThreads;
            if (2 * u < ldr) {
              gl_wait2(px + 2 * u, seq, x[i], y[i], status);
              *reinterpret_cast<float2*>(pg + 2 * u) = make_float2(ll_f(x[i]), ll_f(y[i]));
            }
          }
        }
      }
      __syncthreads();
      reg_trace(prm, tn, TR_X3);
      const int st3 = reinterpret_cast<const int*>(ctl_s + 4)[0];
      if (st3 == 2) { degenerate = true; break; }
      if (!first) {
        lam_new = ctl_s[3];
        rhof = reinterpret_cast<const float*>(ctl_s + 4)[1];
        if (st3 == 1) break;
        lam2 = lam;
        lam = lam_new;
      }
      deferred = reinterpret_cast<const int*>(ctl_s + 1)[1] != 0;
      pscale = reinterpret_cast<const float*>(ctl_s + 2)[0];                   // p = p^/|p^|
      if (!(pscale > 0.f)) { degenerate = true; break; }                      // reading C7
      first = false;
      ++seq;
      ++it;
      // ---- FUSED sweep: t~ = R p (S5), q = R^T t~ (S2 of the next pass), |t~|^2, B-partials (S6) ----
      {
        const unsigned npar = seq & 1u;
        reg_sweep_fused<GT, NV, RPT>(Rr, p_s + (size_t)((it - 1) & 1) * ldr, pscale, ttil_s, qs, red_s, sgrp, ldr);
        reg_trace(prm, tn, TR_SWEEP);
        reg_publish_q<GT>(prm, qs, Qx + (size_t)npar * Gs * G * Ns, b, seq);
        reg_publish_sb(Vb, KV, ttil_s, sgrp, SBx + ((size_t)npar * UB * G + b) * 2, G, NG, mb, k, gsk, seq);
        reg_trace(prm, tn, TR_PUBLISHED);
      }
    }

    // ---- component done ----
    if (degenerate) {
      for (int i = tid; i < NG * RPT; i += kThreads) {
        if (i < mb) Tb[(size_t)k * M + i] = 0.f;
        if (gs) Vb[(size_t)i * KV + k] = 0.f;
      }
      if (owner) {
        for (int i = tid; i < Ns; i += kThreads) {
          if (i < ns) prm.P[(size_t)k * N + n0 + i] = 0.f;
          if (gs) { Pc[(size_t)i * KV + k] = 0.f; Wc[(size_t)i * KV + k] = 0.f; }
        }
      }
      if (b == 0 && tid == 0) { prm.lambda[k] = 0.f; prm.iters[k] = 0; }
      __syncthreads();
    } else {
      const unsigned par = seq & 1u;
      if (gsk && deferred) {
        // ---- final loads (once per component, if S3 was deferred in the pass that converged): p^ = p~ - P_(k) A (S3) of the pass that converged, then
        //      p = p^/|p^| (S4).  The p~ of that pass is in p_s, the owners' A-partials in Ax. ----
        const unsigned fpar = (unsigned)k & 1u, ftag = (unsigned)k + 1u;
        float* pk_w = p_s + (size_t)((it - 1) & 1) * ldr;
        if (owner) {
          reg_gather_a(prm, Ax, (seq - 1u) & 1u, seq - 1u, k, qs, A_s, status);
          for (int i = tid; i < Ns; i += kThreads) praw_s[i] = (i < ns) ? (double)pk_w[n0 + i] : 0.0;   // (its copy for W is in pt_s)
          __syncthreads();
          reg_slice_correct(praw_s, Pc, KV, A_s, ns, k);
          __syncthreads();
          if (w == 0) {
            double q2 = 0.0;
            for (int u = lane; 2 * u < Ns; u += 32) {
              const float v0 = (2 * u < ns) ? (float)praw_s[2 * u] : 0.f;
              const float v1 = (2 * u + 1 < ns) ? (float)praw_s[2 * u + 1] : 0.f;
              gl_st2(Pfx + (size_t)fpar * ldr + n0 + 2 * u, ll_wordf(v0, ftag), ll_wordf(v1, ftag));
              q2 += (double)v0 * (double)v0 + (double)v1 * (double)v1;
            }
            q2 = warp_sum(q2);
            if (lane == 0) gl_st2d(Nfx + (size_t)fpar * (Gs * 2) + (size_t)b * 2, q2, ftag);
          }
        }
        if (tid == (kWarps - 1) * 32) {                                       // arrival hint, as in hop 3
          u64 x = 0, y = 0;
          gl_wait2(Nfx + (size_t)fpar * (Gs * 2) + (size_t)(Gs - 1) * 2, ftag, x, y, status);
        }
        __syncthreads();
        if (w == kWarps - 1) {
          double nsum = 0.0;
          for (int o = lane; o < Gs; o += 32) {
            u64 x0 = 0, y0 = 0;
            gl_wait2(Nfx + (size_t)fpar * (Gs * 2) + (size_t)o * 2, ftag, x0, y0, status);
            nsum += ll_d(x0, y0);
          }
          nsum = warp_sum(nsum);
          if (lane == 0) reinterpret_cast<float*>(ctl_s + 2)[0] = (nsum > 0.0) ? (float)rsqrt(nsum) : 0.f;
        }
        {
          const u64* px = Pfx + (size_t)fpar * ldr;
          for (int u0 = tid; 2 * u0 < ldr; u0 += kThreads * 4) {
            u64 x[4], y[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const int u = u0 + i * kThreads;
              x[i] = 0; y[i] = 0;
              if (2 * u < ldr) gl_ld2(px + 2 * u, x[i], y[i]);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const int u = u0 + i * kThreads;
              if (2 * u < ldr) {
                gl_wait2(px + 2 * u, ftag, x[i], y[i], status);
                *reinterpret_cast<float2*>(pk_w + 2 * u) = make_float2(ll_f(x[i]), ll_f(y[i]));
              }
            }
          }
        }
        __syncthreads();
        pscale = reinterpret_cast<const float*>(ctl_s + 2)[0];
      }
      if (gsk && !owner) {                                                    // everybody needs B for t = t~ - V B
        if (two) {
          const u64* bx = Bx + (size_t)par * (2 + Kpad) * 2;
          for (int e = tid; e < 2 * U; e += kThreads) {
            u64 x = 0, y = 0;
            gl_wait2(bx + 2 * e, seq, x, y, status);
            sb_s[e] = ll_d(x, y);
          }
        } else {
          reg_ll_reduce_all(SBx + ((size_t)par * UB + 1) * G * 2, 2, G * 2, G, (k + 1) >> 1, seq, status, B_s);
        }
        __syncthreads();
      }
      const float lamf = (float)lam_new;
      const float inv = (float)(1.0 / lam_new);
      if (gsk) {                                                              // |B_k|^2 of the finished component (every thread: uniform)
        double bb = 0.0;
        for (int j = 0; j < k; ++j) bb += B_s[j] * B_s[j];
        bf2 += bb * (double)rhof * (double)rhof;
      }
      const float* pk_s = p_s + (size_t)((it - 1) & 1) * ldr;                 // the loads of the last sweep
      // t = t~ - V_(k) B;  GS-PCA: v = t/lambda';  T[:,k] = lambda' v = t (:87,:1037)
      for (int r = w; r < mb; r += kWarps) {
        float c = 0.f;
        if (gsk)
          for (int j = lane; j < k; j += 32) c = fmaf(Vb[(size_t)r * KV + j], (float)B_s[j], c);
        const float corr = (float)warp_sum((double)c);
        if (lane == 0) {
          const float t = (ttil_s[r] - corr) * rhof;                          // (products of the last sweep are short by rho)
          d_s[r] = t;                                                         // S9: R -= lambda' v p^T  /  R -= t p^T
          Tb[(size_t)k * M + r] = prm.out_svd ? t * inv : t;                  // SVD output: the unit vector v
          if (gs) Vb[(size_t)r * KV + k] = t * inv;
        }
      }
      if (owner) {
        for (int i = tid; i < Ns; i += kThreads) {
          const float pk = pk_s[n0 + i] * pscale;
          if (i < ns) prm.P[(size_t)k * N + n0 + i] = pk;
          if (gs) Pc[(size_t)i * KV + k] = pk;
          if (gs && k + 1 < K)                                                // W_k = R_(k+1)^T v_k
            Wc[(size_t)i * KV + k] = (float)(pt_s[i] * (double)rhof / lam_new - lam_new * (double)pk);
        }
      }
      if (b == 0 && tid == 0) { prm.lambda[k] = lamf; prm.iters[k] = it; }
      __syncthreads();
      // ---- S9: rank-1 deflation, in registers (eq. 3) ----
      float4 p4[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        p4[v] = *reinterpret_cast<const float4*>(pk_s + 4 * (gl + GT * v));
        p4[v].x *= pscale; p4[v].y *= pscale; p4[v].z *= pscale; p4[v].w *= pscale;
      }
#pragma unroll
      for (int i = 0; i < RPT; ++i) {
        const float dr = -d_s[g * RPT + i];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          float4 x = Rr.get(i, v);
          axpy4(x, p4[v], dr);
          Rr.set(i, v, x);
        }
      }
    }
    reg_trace(prm, tn, TR_FINAL);
  }
  if (prm.trace_cap > 0 && b == 0 && tid == 0) prm.trace[0] = (unsigned long long)tn;   // (slot 0; the other slots write as many)

  // ---- the residual of eq. (4), back to the row-major workspace ----
#pragma unroll
  for (int i = 0; i < RPT; ++i) {
    const int r = g * RPT + i;
    if (r < mb) {
#pragma unroll
      for (int v = 0; v < NV; ++v) *reinterpret_cast<float4*>(Rb + (size_t)r * ldr + 4 * (gl + GT * v)) = Rr.get(i, v);
    }
  }
}

// Rout[n*M + m] = Rrm[m][n]: the residual in the ABI's column-major layout (no pending deflation).
static __global__ void __launch_bounds__(256) pca_transpose_plain_kernel(const float* __restrict__ Rrm, float* __restrict__ Rout,
                                                                  long long M, int N, int ldr) {
  __shared__ float tile[32][33];
  const long long mt = (long long)blockIdx.x * 32;
  const int nt = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
  for (int j = ty; j < 32; j += 8) {
    const long long m = mt + j;
    const int n = nt + tx;
    tile[j][tx] = (m < M && n < N) ? __ldcg(Rrm + (size_t)m * ldr + n) : 0.f;
  }
  __syncthreads();
#pragma unroll
  for (int j = ty; j < 32; j += 8) {
    const int n = nt + j;
    const long long m = mt + tx;
    if (n < N && m < M) Rout[(size_t)n * M + m] = tile[tx][j];
  }
}

typedef void (*reg_kernel_t)(const RegParams);
// defined in pca_reg_inst*.cu: the compiled (GT, RPT) variants (NV = 2), nullptr if absent
reg_kernel_t reg_kernel_lookup(int GT, int RPT, int RS);

}  // namespace pca
