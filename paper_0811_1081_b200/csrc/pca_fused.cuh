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
//   loop: [hop 1] s, B everywhere -> lambda', test (S7, S8);  slice owners: q slice -> p~ = q - W B, A-partials
//         [hop 2] owners: A -> p^ = p~ - P A, |p^|^2 partials (S3)     (GS-PCA and k > 0 only; taken in the first two passes
//                 of a component and whenever deferring S3 would cost accuracy, see kDeferKappa: otherwise the sweep starts
//                 from p~, |p^|^2 = |p~|^2 - |A|^2 travels with the next exchange and p^ is formed once, at convergence)
//         [hop 3] p = p^/|p^| (or p~/|p~|) everywhere (S4) -> FUSED sweep: t~ = R p (S5), q = R^T t~ (S2 of the
//                 next pass), s = |t~|^2, B-partials = V^T t~ (S6)
//   finalize: [final loads, if S3 was deferred] t = t~ - V B, v = t/lambda', store T, P, lambda, iters, W_k; d <- t
// The hops are NOT grid barriers: data travels between CTAs in self-validating 8-byte words
// {payload, sequence number} (see "LL exchange" below), so a hop costs one store and one polling
// load through L2 (measured: a counter barrier + reduction phase cost 2-6 us, pca_trace).  Every
// CTA takes the same decisions from the same reduced values (fixed summation order, fp64).
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
  int test_mode;         // 0 relative (listings), 1 absolute (text): pca_stagnated()
  int stag2;             // reading C4b: also compare lambda' with the value two passes back (PCA_OPT_STAGNATION)
  int out_svd;           // PCA_OPT_OUTPUT = 1: T holds the unit score vectors V (SVD triple V, U = P, Lambda)
  int defer_s3;          // PCA_OPT_DEFER_S3: 1 = the loads-side Gram-Schmidt may be deferred (kDeferKappa), 0 = never (paper's order)
  int G;                 // CTAs
  int Mb;                // rows per CTA
  int ldr;               // row stride of Rrm / slab (floats) = 4*GT*NV
  int GT;                // threads that share one row (power of two, 32..512)
  int Ns, Gs;            // columns per slice owner, number of owners
  int Kpad;
  // LL exchange buffers: 8-byte words {payload, seq}, double-buffered by sweep parity (see "LL exchange" below)
  unsigned long long* Qx;   // [2][Gs][G][Ns]   partial raw loads, grouped by slice owner
  unsigned long long* SBx;  // [2][G][4 + Kpad] words 0-1: partial |t~|^2 (fp64 bits); words 2-3: this CTA's share of |A|^2
                            //                  (fp64 bits; deferred loads-side Gram-Schmidt, see the kernel); word 4+j: partial B[j]
  unsigned long long* Ax;   // [2][Gs][Kpad]    partial A
  unsigned long long* Px;   // [2][Gs*Ns]       p^ (orthogonalised, not normalised)
  unsigned long long* Nx;   // [2][Gs][2]       partial |p~|^2 (fp64 bits)
  unsigned long long* Pfx;  // [2][Gs*Ns]       final orthogonalised loads p^ of a component (buffer = component parity)
  unsigned long long* Nfx;  // [2][Gs][2]       partial |p^|^2 of the final loads
  float* Pown;              // [Gs][Ns][Kpad]   owner-private panels P[slice, :], W[slice, :] (W = R^T V) when
  float* Wown;              //                  they do not fit in shared memory (cache_pw == 0)
  int cache_pw;
  int Ksm, Mbp;             // shared-memory cache of the CTA's rows of the first Ksm unit score vectors: Vc[Ksm][Mbp]
  unsigned* status;         // [0] != 0: an exchange wait gave up (kSpinLimit)
  unsigned* cnt;            // arrival-counter hints of the three hops, 64 words apart (relaxed; see hop_arrive/hop_wait)
  unsigned long long* trace;  // optional phase trace (PCA_OPT_TRACE): [0] = records written, then records
  int trace_cap;              // capacity in records (0 = off)
  // TMA-staged streaming kernel (pca_tma.cuh, path 7)
  float* Vrm;                 // [M][Kpad] row-major copy of the unit score vectors (helper warps: B-partials during the sweep)
  int SG;                     // ring slots per row group
  int off_ring, off_mbar, off_hb, off_cmd, off_prog;
  // shared-memory carve-up (byte offsets)
  int off_p, off_pdef, off_ttil, off_d, off_qs, off_red, off_sgrp, off_B, off_A, off_scr, off_praw, off_lam, off_pc, off_wc,
      off_slab, off_vc;
};

constexpr int kRB = 4;   // rows per batch
// When may S3 (the loads-side Gram-Schmidt p^ = p~ - P A) be deferred?  Sweeping with p~/|p^| instead of
// p^/|p^| adds  R P_(k) A / |p^| = V_(k) Bm A / |p^|  to t~ (Bm = matrix of the final coefficient vectors B_j of the finished
// components: R_(j+1) p_j = V_(j) B_j).  The scores-side projection removes it exactly, but lambda'^2 = |t~|^2 - |B|^2 is a
// difference: its rounding error grows with |B|^2 / lambda'^2.  The added part is at most |Bm|_F |A| / |p^| long, so a pass
// defers only if the previous pass measured   |A|^2 |Bm|_F^2 <= kDeferKappa |p~|^2 lambda'^2   (added part <= 10 % of lambda':
// no visible cancellation); otherwise, and in the first two passes of a component, it takes the paper's order.
constexpr double kDeferKappa = 1e-2;

// Phase trace (include/pca.h, PCA_OPT_TRACE): thread 0 of CTA 0 appends (phase << 56) | clock64().
enum { TR_COMPONENT = 1, TR_LOADS_DONE = 2, TR_X1 = 3, TR_TEST = 4, TR_QSLICE = 5, TR_APART = 6, TR_X2 = 7,
       TR_PHAT = 8, TR_X3 = 9, TR_PREADY = 10, TR_SWEEP = 11, TR_PUBLISHED = 12, TR_FINAL = 13 };
// BAR.SYNC does not block at issue: a stamp right after __syncthreads() would be the barrier's ISSUE time.  The
// shared-memory read below depends on the barrier's release, and the clock read depends on its value.
__device__ __forceinline__ void trace_mark(const FusedParams& prm, int& tn, int phase) {
  if (prm.trace_cap > 0 && blockIdx.x == 0 && threadIdx.x == 0 && tn < prm.trace_cap) {
    extern __shared__ __align__(16) unsigned char trace_smem_[];
    const unsigned dep = *reinterpret_cast<volatile unsigned*>(trace_smem_);
    unsigned long long c;
    asm volatile("{ .reg .u32 t; and.b32 t, %1, 0; mov.u64 %0, %%clock64; }" : "=l"(c) : "r"(dep) : "memory");
    prm.trace[1 + tn] = ((unsigned long long)phase << 56) | (c & 0x00ffffffffffffffULL);
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
    if (SRC == SRC_GLOBAL && r0 + kRB <= mb) {                          // full batch: no per-row predicates on the loads
      const float* rp = Rb + (size_t)r0 * ldr + 4 * gl;
#pragma unroll
      for (int i = 0; i < kRB; ++i)
#pragma unroll
        for (int v = 0; v < NV; ++v) x[i][v] = ld_stream4(rp + (size_t)i * ldr + 4 * GT * v);
    } else {
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
    }
    float part[kRB];
#pragma unroll
    for (int i = 0; i < kRB; ++i) part[i] = 0.f;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const float4 pv = (SRC == SRC_GLOBAL) ? *reinterpret_cast<const float4*>(p_s + 4 * (gl + GT * v)) : pr[v];
#pragma unroll
      for (int i = 0; i < kRB; ++i) part[i] = dot4(x[i][v], pv, part[i]);
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

// ------------------------------------------------------------------------------------ LL exchange
// Cross-CTA exchange without grid barriers.  Every exchanged 32-bit payload travels in an 8-byte
// word {payload, seq}: the word is written with ONE 64-bit store (single-copy atomic), so a reader
// that sees the expected sequence number also sees the payload -- no fence, no flag, no barrier;
// a hop costs one store and one (polling) load through L2.  seq = number of the sweep that
// produced the data (1, 2, ...; the buffers are zeroed before the launch).  All buffers are
// double-buffered by the parity of seq: a CTA can only be one sweep ahead of the slowest reader
// (it needs the loads p of sweep s+1, which every slice owner publishes only after it has read
// the partials of sweep s from ALL CTAs), so a word of sweep s is never overwritten (by sweep
// s+2) while somebody still waits for it.
// Pairs of words are moved with 16-byte vector accesses (two independent 8-byte atomic halves).
typedef unsigned long long u64;
constexpr unsigned kSpinLimit = 1u << 22;   // polls before a wait gives up and raises status[0] (never in a correct run)

__device__ __forceinline__ u64 ll_word(unsigned payload, unsigned seq) { return ((u64)seq << 32) | (u64)payload; }
__device__ __forceinline__ u64 ll_wordf(float v, unsigned seq) { return ll_word(__float_as_uint(v), seq); }
__device__ __forceinline__ float ll_f(u64 w) { return __uint_as_float((unsigned)w); }
__device__ __forceinline__ void ll_st2(u64* p, u64 a, u64 b) {
  asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ void ll_ld2(const u64* p, u64& a, u64& b) {
  asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}
__device__ __forceinline__ void ll_st2d(u64* p, double v, unsigned seq) {      // one fp64 value in two words (lossless)
  const u64 bits = (u64)__double_as_longlong(v);
  ll_st2(p, ll_word((unsigned)bits, seq), ll_word((unsigned)(bits >> 32), seq));
}
__device__ __forceinline__ double ll_d(u64 a, u64 b) {
  return __longlong_as_double((long long)((b << 32) | (a & 0xffffffffULL)));
}
__device__ __forceinline__ void ll_wait2(const u64* p, unsigned seq, u64& a, u64& b, unsigned* status) {
  unsigned spins = 0;
  while ((unsigned)(a >> 32) != seq || (unsigned)(b >> 32) != seq) {
    ll_ld2(p, a, b);
    if (++spins > kSpinLimit) { *status = 1u; break; }
  }
}

// Arrival hints.  Thousands of threads polling the same words delay the very stores they wait for (measured: 3000-6000
// cycles per hop).  So a producer CTA, after its LL stores, bumps a RELAXED counter, and only thread 0 of a consumer
// CTA polls that counter; the other threads sleep at the block barrier.  The counter orders nothing (no fence): it only
// says "the data is probably there"; the sequence numbers in the data words remain the correctness mechanism.
__device__ __forceinline__ void hop_arrive(unsigned* ctr) {         // call by ONE thread after a block/warp barrier
  asm volatile("red.relaxed.gpu.global.add.u32 [%0], 1;" ::"l"(ctr) : "memory");
}
__device__ __forceinline__ void hop_wait(const unsigned* ctr, unsigned expected, unsigned* status) {
  if (threadIdx.x == 0) {
    unsigned v, spins = 0;
    for (;;) {
      asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
      if ((int)(v - expected) >= 0) break;
      if (++spins > kSpinLimit) { *status = 1u; break; }
    }
  }
  __syncthreads();
}

// ------------------------------------------------------------------------------------ LL words, generic addresses
// Same protocol as pca_fused.cuh ("LL exchange"), but through GENERIC addresses: when the whole problem runs in ONE CTA
// the exchange buffers are placed in shared memory (the warps of the CTA exchange through them exactly as CTAs do through
// L2, at shared-memory latency), otherwise they are the global buffers of the workspace.
__device__ __forceinline__ void gl_st2(u64* p, u64 a, u64 b) {
  asm volatile("st.relaxed.gpu.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ void gl_ld2(const u64* p, u64& a, u64& b) {
  asm volatile("ld.relaxed.gpu.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}
__device__ __forceinline__ void gl_st2d(u64* p, double v, unsigned seq) {
  const u64 bits = (u64)__double_as_longlong(v);
  gl_st2(p, ll_word((unsigned)bits, seq), ll_word((unsigned)(bits >> 32), seq));
}
__device__ __forceinline__ void gl_wait2(const u64* p, unsigned seq, u64& a, u64& b, unsigned* status) {
  unsigned spins = 0;
  while ((unsigned)(a >> 32) != seq || (unsigned)(b >> 32) != seq) {
    gl_ld2(p, a, b);
    if (++spins > kSpinLimit) { *status = 1u; break; }
  }
}

// Owner-side combination of one exchange region: rows of `stride` words, one row per part (= producing CTA), of which the
// first 2*hp words (hp pairs, hp a power of two <= kThreads) are summed over the nparts rows in fp64:
//   out[2*pair], out[2*pair+1] = sum_parts row[part][2*pair], row[part][2*pair+1]          (pairs >= npairs are skipped)
// Thread t owns pair t % hp and the parts t / hp + i * (kThreads / hp) (a warp reads contiguous pairs of a row: coalesced
// 16-byte loads, up to INF in flight per thread), sums them in ascending order, then the threads of a pair are combined
// by shuffles (inside a warp) and through `red` (kThreads double2, across warps) in a fixed order.  If f64_pair0, pair 0
// holds ONE fp64 value.  Two-phase so that two regions can be in flight at once: *_issue, *_finish.
struct RegGather {
  const u64* base;
  int stride, hp, npairs, nparts;
  int f64_pair0;      // the first f64_pair0 pairs hold ONE fp64 value each
  double2* red;       // kThreads entries
  double* out;
};

template <int INF>
__device__ __forceinline__ void reg_gather_issue(const RegGather& gq, u64 (&x)[INF], u64 (&y)[INF]) {
  const int tid = threadIdx.x;
  const int pair = tid & (gq.hp - 1), pslot = tid / gq.hp, pstep = kThreads / gq.hp;
#pragma unroll
  for (int i = 0; i < INF; ++i) {
    const int part = pslot + i * pstep;
    x[i] = 0; y[i] = 0;
    if (part < gq.nparts && pair < gq.npairs) gl_ld2(gq.base + (size_t)part * gq.stride + 2 * pair, x[i], y[i]);
  }
}

template <int INF>
__device__ __forceinline__ void reg_gather_finish(const RegGather& gq, u64 (&x)[INF], u64 (&y)[INF], unsigned seq, unsigned* status) {
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int hp = gq.hp;
  const int pair = tid & (hp - 1), pslot = tid / hp, pstep = kThreads / hp;
  const bool f64 = pair < gq.f64_pair0;
  double a0 = 0.0, a1 = 0.0;
  if (pair < gq.npairs) {
#pragma unroll
    for (int i = 0; i < INF; ++i) {
      const int part = pslot + i * pstep;
      if (part < gq.nparts) {
        gl_wait2(gq.base + (size_t)part * gq.stride + 2 * pair, seq, x[i], y[i], status);
        if (f64) a0 += ll_d(x[i], y[i]);
        else { a0 += (double)ll_f(x[i]); a1 += (double)ll_f(y[i]); }
      }
    }
    for (int p0 = pslot + INF * pstep; p0 < gq.nparts; p0 += INF * pstep) {     // more parts than one batch covers
#pragma unroll
      for (int i = 0; i < INF; ++i) {
        const int part = p0 + i * pstep;
        x[i] = 0; y[i] = 0;
        if (part < gq.nparts) gl_ld2(gq.base + (size_t)part * gq.stride + 2 * pair, x[i], y[i]);
      }
#pragma unroll
      for (int i = 0; i < INF; ++i) {
        const int part = p0 + i * pstep;
        if (part < gq.nparts) {
          gl_wait2(gq.base + (size_t)part * gq.stride + 2 * pair, seq, x[i], y[i], status);
          if (f64) a0 += ll_d(x[i], y[i]);
          else { a0 += (double)ll_f(x[i]); a1 += (double)ll_f(y[i]); }
        }
      }
    }
  }
  for (int o = 16; o >= hp; o >>= 1) {                                        // lanes l and l ^ o own the same pair when o >= hp
    a0 += __shfl_xor_sync(0xffffffffu, a0, o);
    a1 += __shfl_xor_sync(0xffffffffu, a1, o);
  }
  if (hp >= 32) gq.red[tid] = make_double2(a0, a1);
  else if (lane < hp) gq.red[w * hp + lane] = make_double2(a0, a1);
}

// after a __syncthreads(): threads < hp write the sums
__device__ __forceinline__ void reg_gather_store(const RegGather& gq) {
  const int t = threadIdx.x, hp = gq.hp;
  if (t < hp && t < gq.npairs) {
    const int nslots = hp >= 32 ? kThreads / hp : kWarps;
    double a0 = 0.0, a1 = 0.0;
    for (int sl = 0; sl < nslots; ++sl) {
      const double2 v = gq.red[sl * hp + t];
      a0 += v.x; a1 += v.y;
    }
    gq.out[2 * t] = a0;
    gq.out[2 * t + 1] = a1;
  }
}

// One reduction job: out[j] = sum over parts b < nparts of word (base + b*stride)[j], j < 2*units, fp64, fixed order
// (lane l takes parts l, l+32, ... in order, then a shuffle tree).  If f64_unit0, words 0-1 hold one fp64 value.
struct LLJob {
  const u64* base;
  double* out;
  int units, nparts, stride;
  int f64_unit0;      // the first f64_unit0 units hold ONE fp64 value each (words 0-1 of the unit)
};
constexpr int kLLParts = 5;                 // parts per lane held in flight (covers 160 CTAs in one round)

__device__ __forceinline__ void ll_reduce_unit(const LLJob& jb, int u, unsigned seq, unsigned* status) {
  const int lane = threadIdx.x & 31;
  double a0 = 0.0, a1 = 0.0;
  for (int b0 = lane; b0 < jb.nparts; b0 += 32 * kLLParts) {
    u64 x[kLLParts], y[kLLParts];
#pragma unroll
    for (int i = 0; i < kLLParts; ++i) {
      const int bq = b0 + 32 * i;
      x[i] = 0; y[i] = 0;
      if (bq < jb.nparts) ll_ld2(jb.base + (size_t)bq * jb.stride + 2 * u, x[i], y[i]);
    }
#pragma unroll
    for (int i = 0; i < kLLParts; ++i) {
      const int bq = b0 + 32 * i;
      if (bq < jb.nparts) {
        ll_wait2(jb.base + (size_t)bq * jb.stride + 2 * u, seq, x[i], y[i], status);
        if (u < jb.f64_unit0) a0 += ll_d(x[i], y[i]);
        else { a0 += (double)ll_f(x[i]); a1 += (double)ll_f(y[i]); }
      }
    }
  }
  a0 = warp_sum(a0);
  a1 = warp_sum(a1);
  if (lane == 0) { jb.out[2 * u] = a0; jb.out[2 * u + 1] = a1; }
}

// Two jobs share the 16 warps of the CTA (one warp per 2-word unit).  No barrier inside.
__device__ __forceinline__ void ll_reduce2(const LLJob& ja, const LLJob& jb, unsigned seq, unsigned* status) {
  const int w = threadIdx.x >> 5;
  const int total = ja.units + jb.units;
  for (int uu = w; uu < total; uu += kWarps) {
    if (uu < ja.units) ll_reduce_unit(ja, uu, seq, status);
    else ll_reduce_unit(jb, uu - ja.units, seq, status);
  }
}

// Combine the NG group partials of the sweep (fixed order) and publish this CTA's partial raw loads:
// column c of slice owner o = c / Ns goes to Qpar[(o*G + b)*Ns + c % Ns]   (S2)
__device__ __forceinline__ void publish_q_ll(const FusedParams& prm, const float* qs, u64* Qpar, int b, unsigned seq) {
  const int NG = kThreads / prm.GT, ldr = prm.ldr, Ns = prm.Ns;
  const int ncol = prm.Gs * Ns;
  for (int c = threadIdx.x * 2; c < ncol; c += kThreads * 2) {
    float2 a = make_float2(0.f, 0.f);
    if (c < ldr) {
      a = *reinterpret_cast<const float2*>(qs + c);
      for (int g = 1; g < NG; ++g) {
        const float2 v = *reinterpret_cast<const float2*>(qs + (size_t)g * ldr + c);
        a.x += v.x; a.y += v.y;
      }
    }
    const int o = c / Ns, i = c - o * Ns;
    ll_st2(Qpar + ((size_t)o * prm.G + b) * Ns + i, ll_wordf(a.x, seq), ll_wordf(a.y, seq));
  }
}

// praw[i] -= sum_{j<k} C[i*Kpad + j] * coef[j] for the ns columns of this owner (one warp per column).
__device__ __forceinline__ void slice_correct(double* praw_s, const float* C, const double* coef_s, int ns, int k, int Kpad,
                                              int w0 = 0) {                  // warps w0..kWarps-1 take part
  const int lane = threadIdx.x & 31, w = (threadIdx.x >> 5) - w0;
  for (int i = w; i < ns; i += kWarps - w0) {
    const float* ci = C + (size_t)i * Kpad;
    double c = 0.0;
    for (int j = lane; j < k; j += 32) c += (double)ci[j] * coef_s[j];
    c = warp_sum(c);
    if (lane == 0) praw_s[i] -= c;
  }
}

template <int NV, bool RESIDENT>
__global__ void __launch_bounds__(kThreads, 1) pca_fused_kernel(const FusedParams prm) {
  extern __shared__ __align__(16) unsigned char smem[];
  float* p_s = reinterpret_cast<float*>(smem + prm.off_p);        // npx: current unit loads p
  float* pdef_s = reinterpret_cast<float*>(smem + prm.off_pdef);  // ldr: loads of the previous component
  float* ttil_s = reinterpret_cast<float*>(smem + prm.off_ttil);  // Mb : t0 / t~ rows of this CTA
  float* d_s = reinterpret_cast<float*>(smem + prm.off_d);        // Mb : pending deflation vector rows
  float* qs = reinterpret_cast<float*>(smem + prm.off_qs);        // NG x ldr group partials
  float* red_s = reinterpret_cast<float*>(smem + prm.off_red);    // 2 x kWarps x kRB
  double* sgrp = reinterpret_cast<double*>(smem + prm.off_sgrp);  // NG
  double* sb_s = reinterpret_cast<double*>(smem + prm.off_B);     // 4 + Kpad: |t~|^2, -, |A|^2, -, B
  double* B_s = sb_s + 4;
  double* A_s = reinterpret_cast<double*>(smem + prm.off_A);      // Kpad
  double* scr = reinterpret_cast<double*>(smem + prm.off_scr);    // kThreads
  double* ctl_s = scr + kThreads - 8;                             // lambda', decision, 1/|p^| of the current pass
  double* praw_s = reinterpret_cast<double*>(smem + prm.off_praw);// Ns: p~ / p^ slice of this owner
  float* lam_s = reinterpret_cast<float*>(smem + prm.off_lam);    // Kpad
  float* slab = reinterpret_cast<float*>(smem + prm.off_slab);    // resident: Mb x ldr
  float* Vc = reinterpret_cast<float*>(smem + prm.off_vc);        // Ksm x Mbp: cached unit score rows (GS-PCA)

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int b = blockIdx.x;
  const long long M = prm.M;
  const int N = prm.N, K = prm.K, G = prm.G, ldr = prm.ldr, Kpad = prm.Kpad, Ns = prm.Ns, Gs = prm.Gs;
  const int NG = kThreads / prm.GT;
  const int npx = Gs * Ns;                                 // exchanged length of p (>= N)
  const int SBw = 4 + Kpad;
  const bool gs = prm.algo == 1;
  const long long m0 = (long long)b * prm.Mb;
  const int mb = (int)max(0LL, min((long long)prm.Mb, M - m0));
  const int n0 = b * Ns;
  const int ns = max(0, min(Ns, N - n0));
  const bool owner = ns > 0;
  unsigned seq = 0;                                        // sweep number; parity selects the exchange buffers
  unsigned e1 = 0, e2 = 0, e3 = 0, e4 = 0;                 // expected values of the arrival counters
  unsigned* const cnt1 = prm.cnt;
  unsigned* const cnt2 = prm.cnt + 64;
  unsigned* const cnt3 = prm.cnt + 128;
  unsigned* const cnt4 = prm.cnt + 192;
  double* praw2_s = praw_s + Ns;                           // second slice buffer (final p^ of a component)
  unsigned* status = prm.status;
  int tn = 0;                                              // trace records written (thread 0 of CTA 0)
  double bf2 = 0.0;                                        // sum over the finished components of |B_j|^2 (see kDeferKappa)

  float* Rb = prm.Rrm + (size_t)m0 * ldr;
  float* Tb = prm.T + m0;
  // owner-private panels P[slice, 0:k] and W[slice, 0:k] ([Ns][Kpad] floats): shared memory if they fit
  float* Pc = prm.cache_pw ? reinterpret_cast<float*>(smem + prm.off_pc) : prm.Pown + (size_t)b * Ns * Kpad;
  float* Wc = prm.cache_pw ? reinterpret_cast<float*>(smem + prm.off_wc) : prm.Wown + (size_t)b * Ns * Kpad;

  for (int i = tid; i < prm.Mb; i += kThreads) d_s[i] = 0.f;
  for (int n = tid; n < max(ldr, npx); n += kThreads) {
    if (n < npx) p_s[n] = 0.f;
    if (n < ldr) pdef_s[n] = 0.f;
  }
  if (prm.cache_pw)
    for (int i = tid; i < Ns * Kpad; i += kThreads) { Pc[i] = 0.f; Wc[i] = 0.f; }
  for (int i = tid; i < Ns; i += kThreads) praw_s[i] = 0.0;
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
    ++seq;
    {
      const unsigned par = seq & 1u;
      publish_q_ll(prm, qs, prm.Qx + (size_t)par * Gs * G * Ns, b, seq);
      double s = 0.0;
      for (int i = tid; i < mb; i += kThreads) { const double v = (double)ttil_s[i]; s += v * v; }
      s = block_sum(s, scr);                                                    // (block barriers inside: the q stores are issued)
      if (tid == 0) {
        ll_st2d(prm.SBx + ((size_t)par * G + b) * SBw, s, seq);
        hop_arrive(cnt1);
      }
    }
    trace_mark(prm, tn, TR_LOADS_DONE);

    double lam = 0.0, lam2 = 0.0, lam_new = 0.0;
    int it = 0;
    bool degenerate = false;
    bool first = true;
    float inv_pn = 0.f;                                      // 1/|p~| (1/|p^|) of the pass in flight
    bool deferred = false;                                   // the loads of the pass in flight are p~ (S3 deferred), not p^
    for (;;) {
      const unsigned par = seq & 1u;
      // ---- hop 1: |t~|^2 and B (every CTA), raw loads slice (owners) ----
      e1 += (unsigned)G;
      hop_wait(cnt1, e1, status);
      {
        LLJob jq, jsb;
        jq.base = prm.Qx + ((size_t)par * Gs + b) * G * Ns; jq.out = praw_s; jq.units = owner ? (Ns >> 1) : 0;
        jq.nparts = G; jq.stride = Ns; jq.f64_unit0 = false;
        jsb.base = prm.SBx + (size_t)par * G * SBw; jsb.out = sb_s; jsb.units = (gsk && !first) ? 2 + ((k + 1) >> 1) : 1;
        jsb.nparts = G; jsb.stride = SBw; jsb.f64_unit0 = 2;
        if (jsb.units <= 16) {
          ll_reduce2(jsb, jq, seq, status);
        } else {
          // many B units: lanes over the units of a part (contiguous words), parts in turn, instead of a warp per unit with
          // lanes over parts 1 KB apart (measured on config 4 at k = 127: this phase and hop 2 were 10 us each)
          RegGather gsb;
          int hs = 32;
          while (hs < jsb.units) hs <<= 1;
          gsb.base = jsb.base; gsb.stride = SBw; gsb.hp = hs; gsb.npairs = jsb.units; gsb.nparts = G; gsb.f64_pair0 = 2;
          gsb.red = reinterpret_cast<double2*>(qs); gsb.out = sb_s;
          u64 sx[8], sy[8];
          reg_gather_issue<8>(gsb, sx, sy);
          jsb.units = 0;
          ll_reduce2(jsb, jq, seq, status);                                   // the owner's q slice, meanwhile
          reg_gather_finish<8>(gsb, sx, sy, seq, status);
          __syncthreads();
          reg_gather_store(gsb);
        }
      }
      __syncthreads();
      trace_mark(prm, tn, TR_X1);
      // S7/S8 by warp 0 (fp64 sqrt is a long software sequence: once, not 512 times); meanwhile the owners'
      // other warps start on p~ = q - W B, which needs only B.
      if (w == 0) {
        const double s = sb_s[0];
        int st = 0;                                                           // 0 continue, 1 done, 2 degenerate
        double ln = 0.0;
        if (first) {
          if (!(s > 0.0)) st = 2;                                             // zero start column (C7)
        } else {
          double bb = 0.0;
          if (gsk) {                                                          // B = V_(k)^T t~
            for (int j = lane; j < k; j += 32) bb += B_s[j] * B_s[j];
            bb = warp_sum(bb);
          }
          double l2 = s - bb;                                                 // |t~ - V B|^2, V orthonormal
          double rho = 1.0, rho2 = 1.0;
          if (gsk) {
            const double pn2 = ctl_s[3], a2 = sb_s[2];
            if (deferred) {
              // deferred loads-side Gram-Schmidt (see "S3" below): the sweep ran with p~/|p~| instead of p^/|p^|,
              // |p^|^2 = |p~|^2 - |A|^2 (P orthonormal), so every product of the sweep is short of the paper's by
              // rho = |p~|/|p^|
              const double d2 = pn2 - a2;
              if (!(d2 > 0.0)) l2 = 0.0;
              else rho2 = pn2 * fast_rcp(d2);
              l2 *= rho2;
              rho = fast_sqrt(rho2);
            }
            // the NEXT pass defers S3 only if that is harmless (same decision on every CTA): see kDeferKappa
            if (lane == 0) reinterpret_cast<int*>(ctl_s + 4)[0] = (a2 * bf2 <= kDeferKappa * pn2 * lam * lam) ? 1 : 0;
          }
          if (lane == 0) ctl_s[2] = rho;
          if (!(l2 > 0.0)) st = 2;                                            // reading C7
          else {
            ln = fast_sqrt(l2);                                                    // S7
            // S8: listings' strict relative test (reading C3)
            // (+ reading C4b: a period-2 limit cycle of lambda' in fp32 is stagnation too)
            if (pca_stagnated(lam, lam2, ln, prm.eps, prm.test_mode, prm.stag2) || (it >= prm.max_iter)) st = 1;
          }
        }
        if (lane == 0) { ctl_s[0] = ln; reinterpret_cast<int*>(ctl_s + 1)[0] = st; }
      }
      // meanwhile (owners): p~ = q - W B, then the A-partials a_S[j] = sum_{n in S} P[n,j] p~[n] (S3)
      if (owner && gsk && w > 0) {
        if (!first) {
          slice_correct(praw_s, Wc, B_s, ns, k, Kpad, 1);
          named_bar_sync(1, kThreads - 32);                                   // warps 1..15 (warp 0 is busy with the test)
        }
        const int u = tid - 32;                                               // warps 1..15: one thread per pair of A
        for (int j0 = 2 * u; j0 < k; j0 += 2 * (kThreads - 32)) {
          double a0 = 0.0, a1 = 0.0;
          for (int i = 0; i < ns; ++i) {
            const float2 pj = *reinterpret_cast<const float2*>(Pc + (size_t)i * Kpad + j0);
            a0 += (double)pj.x * praw_s[i];
            a1 += (double)pj.y * praw_s[i];
          }
          if (j0 + 1 >= k) a1 = 0.0;
          ll_st2(prm.Ax + ((size_t)par * Gs + b) * Kpad + j0, ll_wordf((float)a0, seq), ll_wordf((float)a1, seq));
        }
      }
      __syncthreads();
      const int st = reinterpret_cast<const int*>(ctl_s + 1)[0];
      if (st == 2) { degenerate = true; break; }
      bool done = false;
      if (!first) {
        lam_new = ctl_s[0];
        done = st == 1;
        if (!done) { lam2 = lam; lam = lam_new; }
      }
      trace_mark(prm, tn, TR_TEST);
      if (done) break;
      trace_mark(prm, tn, TR_QSLICE);

      // ---- S3, deferred.  The paper orthogonalises the loads first, p^ = p~ - P_(k) A, and multiplies
      // then, t~ = R p^.  R P_(k) lies in span V_(k) (deflation: R_(j+1) p_j = t~_j - t_j = V_(j) B_j, and later deflations
      // add multiples of v_i), and the scores-side projection t = t~ - V_(k) V_(k)^T t~ removes that
      // span, so R p~ and R p^ give the SAME t: the sweep can start from p~ without waiting for A = sum of the owners'
      // partials (one dependent cross-CTA hop less per pass).  What the iteration needs from A is |p^|^2 = |p~|^2 - |A|^2
      // (lambda' scales with 1/|p^|); it travels with the NEXT exchange.  p^ itself is formed once, when the component has
      // converged ("final loads" below).  (The two-sweep kernel keeps the paper's literal order.)
      // Deferring costs accuracy when A is NOT small (the first pass of a component starts from a raw column; fixed-pass
      // runs never converge): t~ then carries a large component in span V_(k) and lambda'^2 = |t~|^2 - |B|^2 cancels.  So the
      // first two passes of a component, and every pass for which the bound of kDeferKappa fails, take the paper's order.
      const bool defer_now = prm.defer_s3 != 0 && gsk && !first && reinterpret_cast<const int*>(ctl_s + 4)[0] != 0;
      if (gsk && owner && tid == 0) hop_arrive(cnt2);                         // A-partials of this pass are out
      trace_mark(prm, tn, TR_APART);
      if (gsk) e2 += (unsigned)Gs;
      if (gsk && owner && !defer_now) {
        hop_wait(cnt2, e2, status);
        // ---- hop 2: A = sum of the owners' partials;  p^ = p~ - P_(k) A ----
        if (k <= 30) {
          LLJob ja, jn;
          ja.base = prm.Ax + (size_t)par * Gs * Kpad; ja.out = A_s; ja.units = (k + 1) >> 1; ja.nparts = Gs; ja.stride = Kpad;
          ja.f64_unit0 = 0;
          jn = ja; jn.units = 0;
          ll_reduce2(ja, jn, seq, status);
        } else {
          RegGather ga;
          const int ua = (k + 1) >> 1;
          int ha = 32;
          while (ha < ua) ha <<= 1;
          ga.base = prm.Ax + (size_t)par * Gs * Kpad; ga.stride = Kpad; ga.hp = ha; ga.npairs = ua; ga.nparts = Gs;
          ga.f64_pair0 = 0; ga.red = reinterpret_cast<double2*>(qs); ga.out = A_s;
          u64 ax8[8], ay8[8];
          reg_gather_issue<8>(ga, ax8, ay8);
          reg_gather_finish<8>(ga, ax8, ay8, seq, status);
          __syncthreads();
          reg_gather_store(ga);
        }
        __syncthreads();
        trace_mark(prm, tn, TR_X2);
        slice_correct(praw_s, Pc, A_s, ns, k, Kpad);
        __syncthreads();
      }
      deferred = defer_now;
      // ---- publish the p~ slice and its squared norm (S4, first half) ----
      if (owner && w == 0) {
        double q2 = 0.0;
        for (int u = lane; 2 * u < Ns; u += 32) {
          const float v0 = (2 * u < ns) ? (float)praw_s[2 * u] : 0.f;
          const float v1 = (2 * u + 1 < ns) ? (float)praw_s[2 * u + 1] : 0.f;
          ll_st2(prm.Px + (size_t)par * npx + n0 + 2 * u, ll_wordf(v0, seq), ll_wordf(v1, seq));
          q2 += (double)v0 * (double)v0 + (double)v1 * (double)v1;
        }
        q2 = warp_sum(q2);
        if (lane == 0) {
          ll_st2d(prm.Nx + ((size_t)par * Gs + b) * 2, q2, seq);
          hop_arrive(cnt3);                                                   // (the warp's p^ stores precede it in program order)
        }
      }
      trace_mark(prm, tn, TR_PHAT);
      e3 += (unsigned)Gs;
      hop_wait(cnt3, e3, status);
      // ---- hop 3: gather p^ and |p^|^2 ----
      if (w == kWarps - 1) {
        LLJob jn;
        jn.base = prm.Nx + (size_t)par * Gs * 2; jn.out = scr; jn.units = 1; jn.nparts = Gs; jn.stride = 2; jn.f64_unit0 = true;
        ll_reduce_unit(jn, 0, seq, status);
        __syncwarp();
        if (lane == 0) {
          ctl_s[3] = scr[0];                                                  // |p~|^2
          reinterpret_cast<float*>(ctl_s + 1)[1] = (scr[0] > 0.0) ? (float)rsqrt(scr[0]) : 0.f;
        }
      }
      if (gsk && w == kWarps - 2) {
        // this CTA's share of |A|^2: the entries A[2u], A[2u+1] of its units u = b, b + G, ... summed over the owners'
        // partials (fixed order); published with |t~|^2 after the sweep, summed over the CTAs at the next hop 1
        double a2 = 0.0;
        LLJob ja;
        ja.base = prm.Ax + (size_t)par * Gs * Kpad; ja.out = scr + 8; ja.nparts = Gs; ja.stride = Kpad; ja.f64_unit0 = 0;
        ja.units = (k + 1) >> 1;
        double* ao = scr + 8;                                                  // (scr[0..] belongs to the norm warp)
        for (int u = b; u < ja.units; u += G) {
          ja.out = ao - 2 * u;                                                // the unit's two sums land in ao[0], ao[1]
          ll_reduce_unit(ja, u, seq, status);
          __syncwarp();
          a2 += ao[0] * ao[0] + ao[1] * ao[1];
          __syncwarp();
        }
        if (lane == 0) scr[4] = a2;
      }
      {
        const u64* px = prm.Px + (size_t)par * npx;
        for (int u0 = tid; 2 * u0 < npx; u0 += kThreads * 4) {
          u64 x[4], y[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int u = u0 + i * kThreads;
            x[i] = 0; y[i] = 0;
            if (2 * u < npx) ll_ld2(px + 2 * u, x[i], y[i]);
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int u = u0 + i * kThreads;
            if (2 * u < npx) {
              ll_wait2(px + 2 * u, seq, x[i], y[i], status);
              *reinterpret_cast<float2*>(p_s + 2 * u) = make_float2(ll_f(x[i]), ll_f(y[i]));
            }
          }
        }
      }
      __syncthreads();
      trace_mark(prm, tn, TR_X3);
      inv_pn = reinterpret_cast<const float*>(ctl_s + 1)[1];                  // p = p~/|p~| (see S3 above)
      const double a2mine = gsk ? scr[4] : 0.0;
      if (!(inv_pn > 0.f)) { degenerate = true; break; }                      // reading C7
      for (int n = tid; n < npx; n += kThreads) p_s[n] *= inv_pn;             // each thread rescales what it wrote
      __syncthreads();
      first = false;
      trace_mark(prm, tn, TR_PREADY);
      // ---- FUSED sweep: t~ = R p (S5), q = R^T t~, s = |t~|^2 ----
      ++seq;
      ++it;
      {
        const unsigned npar = seq & 1u;
        const bool rev = (seq & 1u) != 0;
        const long long tsw0 = (prm.trace_cap > 0 && tid == 0) ? clock64() : 0;
        if constexpr (RESIDENT) sweep_fused<NV, SRC_SLAB>(prm, Rb, slab, mb, p_s, ttil_s, qs, red_s, sgrp, false);
        else                    sweep_fused<NV, SRC_GLOBAL>(prm, Rb, slab, mb, p_s, ttil_s, qs, red_s, sgrp, rev);
        if (prm.trace_cap > 0 && tid == 0) {                                  // per-CTA sweep cycles and SM id, after the records
          unsigned smid;
          asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
          prm.trace[1 + prm.trace_cap + b] += (unsigned long long)(clock64() - tsw0);
          prm.trace[1 + prm.trace_cap + G + b] = smid;
        }
        trace_mark(prm, tn, TR_SWEEP);
        publish_q_ll(prm, qs, prm.Qx + (size_t)npar * Gs * G * Ns, b, seq);
        u64* sbx = prm.SBx + ((size_t)npar * G + b) * SBw;
        if (tid == 0) {
          double a = 0.0;
          for (int g = 0; g < NG; ++g) a += sgrp[g];
          ll_st2d(sbx, a, seq);
          if (gsk) ll_st2d(sbx + 2, a2mine, seq);
        }
        __syncthreads();   // (measured: without this barrier the B-partial loop below runs 2-6 x slower -- warp 0 enters it
                           //  diverged from the tid == 0 block above and its full-mask shuffles pay for it every iteration)
        if (gsk) {                                                            // S6: B-partials V^T t~
          // the CTA's rows of the first Ksm unit score vectors are cached in shared memory (Vc, column-major), the rest
          // comes from T in global memory (L2)
          for (int j0 = 2 * w; j0 < k; j0 += 2 * kWarps) {
            const bool two = j0 + 1 < k;
            float a0 = 0.f, a1 = 0.f;
            if (j0 + 1 < prm.Ksm) {
              const float* c0 = Vc + (size_t)j0 * prm.Mbp;
              const float* c1 = c0 + prm.Mbp;
              for (int i = lane; i < mb; i += 32) {
                const float tt = ttil_s[i];
                a0 = fmaf(c0[i], tt, a0);
                if (two) a1 = fmaf(c1[i], tt, a1);
              }
            } else {
              const float* v0 = Tb + (size_t)j0 * M;
              const float* v1 = v0 + M;
              for (int i = lane; i < mb; i += 32) {
                const float tt = ttil_s[i];
                a0 = fmaf(v0[i], tt, a0);
                if (two) a1 = fmaf(v1[i], tt, a1);
              }
            }
            const double s0 = warp_sum((double)a0), s1 = warp_sum((double)a1);
            if (lane == 0) ll_st2(sbx + 4 + j0, ll_wordf((float)s0, seq), ll_wordf((float)s1, seq));
          }
        }
        __syncthreads();                                                      // all LL stores of this CTA are issued
        if (tid == 0) hop_arrive(cnt1);
        trace_mark(prm, tn, TR_PUBLISHED);
      }
    }

    if (!degenerate && gsk && deferred) {
      // ---- final loads (once per component, if the pass that converged had S3 deferred): p^ = p~ - P_(k) A (S3) of the pass that converged,
      //      p = p^/|p^| (S4).  p_s holds p~/|p~|, the owners' A-partials of that pass are in Ax. ----
      const unsigned apar = (seq - 1u) & 1u, aseq = seq - 1u;
      const unsigned fpar = (unsigned)k & 1u, ftag = (unsigned)k + 1u;
      if (owner) {
        if (k <= 30) {
          LLJob ja, jn;
          ja.base = prm.Ax + (size_t)apar * Gs * Kpad; ja.out = A_s; ja.units = (k + 1) >> 1; ja.nparts = Gs; ja.stride = Kpad;
          ja.f64_unit0 = 0;
          jn = ja; jn.units = 0;
          ll_reduce2(ja, jn, aseq, status);
        } else {
          RegGather ga;
          const int ua = (k + 1) >> 1;
          int ha = 32;
          while (ha < ua) ha <<= 1;
          ga.base = prm.Ax + (size_t)apar * Gs * Kpad; ga.stride = Kpad; ga.hp = ha; ga.npairs = ua; ga.nparts = Gs;
          ga.f64_pair0 = 0; ga.red = reinterpret_cast<double2*>(qs); ga.out = A_s;
          u64 ax8[8], ay8[8];
          reg_gather_issue<8>(ga, ax8, ay8);
          reg_gather_finish<8>(ga, ax8, ay8, aseq, status);
          __syncthreads();
          reg_gather_store(ga);
        }
        __syncthreads();
        for (int i = tid; i < Ns; i += kThreads) praw2_s[i] = (i < ns) ? (double)p_s[n0 + i] : 0.0;
        for (int j = tid; j < k; j += kThreads) A_s[j] *= (double)inv_pn;   // A of the scaled vector p~/|p~|
        __syncthreads();
        slice_correct(praw2_s, Pc, A_s, ns, k, Kpad);
        __syncthreads();
        if (w == 0) {
          double q2 = 0.0;
          for (int u = lane; 2 * u < Ns; u += 32) {
            const float v0 = (2 * u < ns) ? (float)praw2_s[2 * u] : 0.f;
            const float v1 = (2 * u + 1 < ns) ? (float)praw2_s[2 * u + 1] : 0.f;
            ll_st2(prm.Pfx + (size_t)fpar * npx + n0 + 2 * u, ll_wordf(v0, ftag), ll_wordf(v1, ftag));
            q2 += (double)v0 * (double)v0 + (double)v1 * (double)v1;
          }
          q2 = warp_sum(q2);
          if (lane == 0) {
            ll_st2d(prm.Nfx + ((size_t)fpar * Gs + b) * 2, q2, ftag);
            hop_arrive(cnt4);
          }
        }
      }
      e4 += (unsigned)Gs;
      hop_wait(cnt4, e4, status);
      if (w == kWarps - 1) {
        LLJob jn;
        jn.base = prm.Nfx + (size_t)fpar * Gs * 2; jn.out = scr; jn.units = 1; jn.nparts = Gs; jn.stride = 2; jn.f64_unit0 = 1;
        ll_reduce_unit(jn, 0, ftag, status);
        __syncwarp();
        if (lane == 0) reinterpret_cast<float*>(ctl_s + 1)[1] = (scr[0] > 0.0) ? (float)rsqrt(scr[0]) : 0.f;
      }
      {
        const u64* px = prm.Pfx + (size_t)fpar * npx;
        for (int u0 = tid; 2 * u0 < npx; u0 += kThreads * 4) {
          u64 x[4], y[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int u = u0 + i * kThreads;
            x[i] = 0; y[i] = 0;
            if (2 * u < npx) ll_ld2(px + 2 * u, x[i], y[i]);
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int u = u0 + i * kThreads;
            if (2 * u < npx) {
              ll_wait2(px + 2 * u, ftag, x[i], y[i], status);
              *reinterpret_cast<float2*>(p_s + 2 * u) = make_float2(ll_f(x[i]), ll_f(y[i]));
            }
          }
        }
      }
      __syncthreads();
      const float inv_f = reinterpret_cast<const float*>(ctl_s + 1)[1];
      for (int n = tid; n < npx; n += kThreads) p_s[n] *= inv_f;
      __syncthreads();
    }
    // ---- component done ----
    if (degenerate) {
      for (int i = tid; i < mb; i += kThreads) {
        Tb[(size_t)k * M + i] = 0.f; d_s[i] = 0.f;
        if (gs && k < prm.Ksm) Vc[(size_t)k * prm.Mbp + i] = 0.f;
      }
      if (tid < ns) prm.P[(size_t)k * N + n0 + tid] = 0.f;
      if (tid < Ns) { Pc[(size_t)tid * Kpad + k] = 0.f; Wc[(size_t)tid * Kpad + k] = 0.f; }
      for (int n = tid; n < ldr; n += kThreads) pdef_s[n] = 0.f;
      if (b == 0 && tid == 0) { prm.lambda[k] = 0.f; prm.iters[k] = 0; }
      if (tid == 0) lam_s[k] = 0.f;
    } else {
      const float lamf = (float)lam_new;
      const float inv = (float)(1.0 / lam_new);
      const double rho = (gsk && deferred) ? ctl_s[2] : 1.0;                               // products of the last sweep are short by rho (S3)
      const float rhof = (float)rho;
      if (gsk) {                                                              // |B_k|^2 of the finished component (every thread: uniform)
        double bb = 0.0;
        for (int j = 0; j < k; ++j) bb += B_s[j] * B_s[j];
        bf2 += bb * rho * rho;
      }
      // t = t~ - V_(k) B;  GS-PCA: v = t/lambda'
      for (int i = tid; i < mb; i += kThreads) {
        float t = ttil_s[i];
        if (gsk) {
          float corr = 0.f;
          for (int j = 0; j < k; ++j) corr = fmaf(Tb[(size_t)j * M + i], (float)B_s[j], corr);
          t = (t - corr) * rhof;
        }
        d_s[i] = t;                                                           // R -= lambda v p^T  /  R -= t p^T
        Tb[(size_t)k * M + i] = (gs || prm.out_svd) ? t * inv : t;
        if (gs && k < prm.Ksm) Vc[(size_t)k * prm.Mbp + i] = t * inv;
      }
      if (tid < ns) {
        const float pk = p_s[n0 + tid];
        prm.P[(size_t)k * N + n0 + tid] = pk;
        Pc[(size_t)tid * Kpad + k] = pk;
        if (gs && k + 1 < K)                                                  // W_k = R_(k+1)^T v_k
          Wc[(size_t)tid * Kpad + k] = (float)(praw_s[tid] * rho / lam_new - lam_new * (double)pk);
      }
      for (int n = tid; n < ldr; n += kThreads) pdef_s[n] = (n < npx) ? p_s[n] : 0.f;
      if (b == 0 && tid == 0) { prm.lambda[k] = lamf; prm.iters[k] = it; }
      if (tid == 0) lam_s[k] = lamf;
    }
    __syncthreads();
    trace_mark(prm, tn, TR_FINAL);
  }
  if (prm.trace_cap > 0 && b == 0 && tid == 0) prm.trace[0] = (unsigned long long)tn;

  // resident: hand the slab back (the last deflation is applied by pca_transpose_out_kernel)
  if constexpr (RESIDENT) sweep_loads<NV, SRC_SLAB, DST_GLOBAL, false, false>(prm, Rb, slab, mb, ttil_s, d_s, pdef_s, qs);
  // ---- S10: GS-PCA  T <- V Lambda; skipped for the SVD output V, U, Lambda ----
  if (gs && !prm.out_svd) {
    __syncthreads();
    for (int kk = 0; kk < K; ++kk) {
      const float l = lam_s[kk];
      for (int i = tid; i < mb; i += kThreads) Tb[(size_t)kk * M + i] *= l;
    }
  }
}

// ------------------------------------------------------------------------------------ transposes
// Rrm[m][n] = X[n*M + m] for n < N, 0 for N <= n < ldr                      (R <- X)
static __global__ void __launch_bounds__(256) pca_transpose_in_kernel(const float* __restrict__ X, float* __restrict__ Rrm,
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
// dscale != nullptr (SVD output: T holds unit vectors): d is scaled by dscale[0] = lambda[K-1].
static __global__ void __launch_bounds__(256) pca_transpose_out_kernel(const float* __restrict__ Rrm, float* __restrict__ Rout,
                                                                const float* __restrict__ d, const float* __restrict__ p,
                                                                const float* __restrict__ dscale, long long M, int N, int ldr) {
  __shared__ float tile[32][33];
  const long long mt = (long long)blockIdx.x * 32;
  const int nt = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const float ds = dscale ? __ldcg(dscale) : 1.f;
#pragma unroll
  for (int j = ty; j < 32; j += 8) {
    const long long m = mt + j;
    const int n = nt + tx;
    float v = 0.f;
    if (m < M && n < N) v = fmaf(-__ldcg(d + m) * ds, __ldcg(p + n), __ldcg(Rrm + (size_t)m * ldr + n));
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
