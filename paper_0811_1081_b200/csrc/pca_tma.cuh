// =====================================================================================
// pca_tma.cuh -- TMA-staged single-sweep streaming kernel (path 7; north_star (e): "falling back to
// TMA-staged HBM streaming when [R] does not [fit on chip]").
//
// Same iteration, same exchange chain and same arithmetic as pca_fused_kernel<NV, false> (pca_fused.cuh; the
// paper's gemv pair t = R p, p' = R^T t of PAPER.md:1028,:1023 / :564,:562 taken from ONE read of R per inner
// pass), but the rows of R do not travel through the register file / L1 on their way in:
//
//   * every row group (GT threads that share a row) owns a private RING of SG slots in shared memory; a slot holds
//     one batch of RB consecutive rows (RB*ldr floats, contiguous in the row-major residual), filled by ONE
//     bulk-async copy (cp.async.bulk.shared.global, SASS UBLKCP) that completes on the slot's mbarrier.  The group
//     refills a slot itself as soon as its threads have pulled the batch into registers, so SG batches per group are
//     always in flight or ready -- across the END of a sweep too: the batches of the NEXT sweep (run in the opposite
//     row order, so that its first rows are the L2-hot tail of this one) are already on their way while the CTA
//     sits in the cross-CTA exchange chain (hops 1-3), when the plain-load kernel keeps HBM idle;
//   * bulk copies need no L1 lines, so the whole 227 KB can be shared memory (the plain-load kernel had to stay
//     below 100 KB: its 128 KB of loads in flight per SM live in L1);
//   * the Gram-Schmidt coefficients B = V_(k)^T t~ (S6) are accumulated DURING the sweep by kHelperWarps
//     extra warps from a row-major copy Vrm of the unit score vectors: they follow the row groups batch by batch
//     (progress words in shared memory), so that only the last batch is left when the sweep ends (plain-load
//     kernel: a separate phase over the 4kM-byte panel after every sweep, 10 us at k = 127 on config 4).
//
// A sweep that WRITES R (the fused deflation of S9, once per component) must not be overtaken by copies of the next
// sweep: refills stop at the end of such a sweep, every thread orders its stores before later async-proxy reads
// (fence.proxy.async), the CTA synchronises, then the ring is topped up.
// =====================================================================================
#pragma once
#include "pca_fused.cuh"

namespace pca {

constexpr int kHelperWarps = 4;   // warps 16..19: one per SM sub-partition (any 17th warp already lowers the register cap to 96)
constexpr int kTmaThreads = kThreads + 32 * kHelperWarps;
enum { BAR_CTA = 0, BAR_HSTART = 14, BAR_HDONE = 15 };           // named barriers 1..NG: row groups (named_bar_sync)
enum { HCMD_EXIT = 0, HCMD_SWEEP = 1 };

// the kThreads compute threads only (the helper warps never take part in barrier 0)
__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0, %0;" ::"n"(kThreads) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(void* bar, unsigned parity) {
  unsigned ok;
  asm volatile(
      "{\n\t.reg .pred P1;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, P1;\n\t}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return ok != 0;
}
// (try_wait suspends the thread for a hardware time slice; like every other wait of the kernel this one gives up after
//  kSpinLimit polls and raises the status word instead of hanging the GPU -- never in a correct run)
__device__ __forceinline__ void mbar_wait(void* bar, unsigned parity, unsigned* status) {
  unsigned spins = 0;
  while (!mbar_try_wait(bar, parity)) {
    if (++spins > kSpinLimit) { *status = 1u; break; }
  }
}
// one contiguous block global -> shared, completion (bytes) on an mbarrier of this CTA             (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, void* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void st_release_cta(unsigned* p, unsigned v) {
  asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned ld_acquire_cta(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
  return v;
}

// block_sum / hop_wait of the plain-load kernel with the compute-threads barrier
__device__ __forceinline__ double block_sum_c(double v, double* scr) {
  v = warp_sum(v);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  cta_sync();
  if (lane == 0) scr[w] = v;
  cta_sync();
  if (w == 0) {
    double s = (lane < kWarps) ? scr[lane] : 0.0;
    s = warp_sum(s);
    if (lane == 0) scr[kWarps] = s;
  }
  cta_sync();
  return scr[kWarps];
}
__device__ __forceinline__ void hop_wait_c(const unsigned* ctr, unsigned expected, unsigned* status) {
  if (threadIdx.x == 0) {
    unsigned v, spins = 0;
    for (;;) {
      asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
      if ((int)(v - expected) >= 0) break;
      if (++spins > kSpinLimit) { *status = 1u; break; }
    }
  }
  cta_sync();
}

// ------------------------------------------------------------------------------------ ring of one row group
// Batch stream of group g: sweep 0 batches, sweep 1 batches, ...; within sweep `sw` the group takes the batch
// positions bq = g, g + NG, ... < nb and position bq is row batch bi = (sw odd) ? nb-1-bq : bq (alternate sweeps run
// in opposite row order).  `cons` / `iss` count consumed / issued batches of the stream (slot = count % SG, the
// mbarrier phase parity = (count / SG) & 1).  All threads of the group keep `cons`; the group leader keeps the rest.
template <int RB>
struct Ring {
  float* slots;             // SG slots of RB*ldr floats
  unsigned long long* full; // SG mbarriers
  const float* Rb;          // the CTA's rows of the row-major residual
  int SG, ldr, mb, nb, g, NG;
  unsigned* status;
  // running indices instead of count % SG, count / SG (integer division is a long serial sequence on the leader's path)
  int cons_slot;            // slot of the next batch to consume (all threads of the group)
  unsigned cons_par;        // its mbarrier phase parity
  unsigned cons;            // batches consumed
  int iss_slot;             // leader: slot of the next batch to issue
  int inflight;             // leader: issued and not yet consumed
  int iss_sw, iss_bq;       // leader: stream position of the next batch to issue

  __device__ __forceinline__ const float* cur_slot() const { return slots + (size_t)cons_slot * (RB * ldr); }
  __device__ __forceinline__ void wait_next() const { mbar_wait(full + cons_slot, cons_par, status); }   // batch has landed
  __device__ __forceinline__ void consumed() {                             // all threads of the group, after the batch is in registers
    ++cons;
    if (++cons_slot == SG) { cons_slot = 0; cons_par ^= 1u; }
  }
  // leader: issue copies while a slot is free and the stream position is within sweeps <= limit_sw
  __device__ __forceinline__ void top_up(int limit_sw) {
    while (inflight < SG && iss_sw <= limit_sw && g < nb) {
      const int bi = (iss_sw & 1) ? (nb - 1 - iss_bq) : iss_bq;
      const int r0 = bi * RB;
      const int rows = min(RB, mb - r0);
      const unsigned bytes = (unsigned)rows * (unsigned)ldr * 4u;
      unsigned long long* bar = full + iss_slot;
      mbar_expect_tx(bar, bytes);
      bulk_g2s(slots + (size_t)iss_slot * (RB * ldr), Rb + (size_t)r0 * ldr, bytes, bar);
      ++inflight;
      if (++iss_slot == SG) iss_slot = 0;
      iss_bq += NG;
      if (iss_bq >= nb) { iss_bq = g; ++iss_sw; }
    }
  }
};

// sum over the GT threads of a row group of RB values per thread; every thread gets all RB sums.
// Butterfly inside the warp (row i ends up in the lanes [i*32/RB, (i+1)*32/RB)), then (WG > 1 warps per group) one
// shared-memory exchange under the group's named barrier.
template <int RB>
__device__ __forceinline__ void group_row_sums(float (&part)[RB], float (&tt)[RB], int WG, int g, int GT, int wg, int lane,
                                               float* red_s, int& parity) {
  float kk;
  if constexpr (RB == 4) {
    const bool hi = (lane & 16) != 0;
    float k0 = hi ? part[2] : part[0], k1 = hi ? part[3] : part[1];
    const float s0 = hi ? part[0] : part[2], s1 = hi ? part[1] : part[3];
    k0 += __shfl_xor_sync(0xffffffffu, s0, 16);
    k1 += __shfl_xor_sync(0xffffffffu, s1, 16);
    const bool h8 = (lane & 8) != 0;
    kk = h8 ? k1 : k0;
    const float ss = h8 ? k0 : k1;
    kk += __shfl_xor_sync(0xffffffffu, ss, 8);
    kk += __shfl_xor_sync(0xffffffffu, kk, 4);
  } else if constexpr (RB == 2) {
    const bool hi = (lane & 16) != 0;
    kk = hi ? part[1] : part[0];
    const float ss = hi ? part[0] : part[1];
    kk += __shfl_xor_sync(0xffffffffu, ss, 16);
    kk += __shfl_xor_sync(0xffffffffu, kk, 8);
    kk += __shfl_xor_sync(0xffffffffu, kk, 4);
  } else {
    kk = part[0];
    kk += __shfl_xor_sync(0xffffffffu, kk, 16);
    kk += __shfl_xor_sync(0xffffffffu, kk, 8);
    kk += __shfl_xor_sync(0xffffffffu, kk, 4);
  }
  kk += __shfl_xor_sync(0xffffffffu, kk, 2);
  kk += __shfl_xor_sync(0xffffffffu, kk, 1);
  constexpr int LPR = 32 / RB;                                             // lanes per row after the butterfly
  if (WG == 1) {
#pragma unroll
    for (int i = 0; i < RB; ++i) tt[i] = __shfl_sync(0xffffffffu, kk, LPR * i);
    __syncwarp();
  } else {
    float* rs = red_s + (size_t)parity * (kWarps * RB) + (size_t)(g * WG) * RB;
    if ((lane & (LPR - 1)) == 0) rs[wg * RB + lane / LPR] = kk;
    named_bar_sync(1 + g, GT);
#pragma unroll
    for (int i = 0; i < RB; ++i) tt[i] = 0.f;
    for (int w = 0; w < WG; ++w) {
#pragma unroll
      for (int i = 0; i < RB; ++i) tt[i] += rs[w * RB + i];
    }
    parity ^= 1;
  }
}

// ------------------------------------------------------------------------------------ FUSED sweep from the ring
// For every owned row r:  t~[r] = sum_n R[r,n] p[n]  (S5);  q[n] += R[r,n] t~[r]  (S2 of the next
// pass).  A batch is pulled from its ring slot into registers (RB rows x NV float4 per thread), the
// RB partial dots are reduced over the group, the slot is handed back (refill) and the registers are used again for
// the second product.  Leaves qs[g][ldr], ttil_s[rows], sgrp[g] = sum t~^2 (fp64); ends with cta_sync().
template <int NV, int RB>
__device__ __forceinline__ void sweep_fused_ring(const FusedParams& prm, Ring<RB>& rg, int sw, const float* p_s,
                                                 float* ttil_s, float* qs, float* red_s, double* sgrp, unsigned* prog_s) {
  const int GT = prm.GT, NG = kThreads / GT, WG = GT >> 5, ldr = prm.ldr;
  const int tid = threadIdx.x, g = tid / GT, gl = tid - g * GT, lane = tid & 31, wg = gl >> 5;
  float4 q[NV];                                                            // (p is re-read from shared memory per batch:
#pragma unroll                                                             //  16 registers less, no spills in the loop)
  for (int v = 0; v < NV; ++v) q[v] = make_float4(0.f, 0.f, 0.f, 0.f);
  double sacc = 0.0;
  int parity = 0;
  const bool rev = (sw & 1) != 0;
  const int gl2 = GT >= 64 ? 32 : 0;                                      // thread of the group that records t~ and |t~|^2
  for (int bq = g; bq < rg.nb; bq += NG) {
    const int bi = rev ? (rg.nb - 1 - bq) : bq;
    const int r0 = bi * RB;
    const int rows = min(RB, rg.mb - r0);
    rg.wait_next();
    const float* sl = rg.cur_slot();
    float4 x[RB][NV];
#pragma unroll
    for (int i = 0; i < RB; ++i) {
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        if (i < rows) x[i][v] = *reinterpret_cast<const float4*>(sl + (size_t)i * ldr + 4 * (gl + GT * v));
        else x[i][v] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
    float part[RB], tt[RB];
#pragma unroll
    for (int i = 0; i < RB; ++i) part[i] = 0.f;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const float4 pv = *reinterpret_cast<const float4*>(p_s + 4 * (gl + GT * v));
#pragma unroll
      for (int i = 0; i < RB; ++i) part[i] = dot4(x[i][v], pv, part[i]);
    }
    group_row_sums<RB>(part, tt, WG, g, GT, wg, lane, red_s, parity);     // every thread of the group has read the slot
    rg.consumed();
    if (gl == 0) {
      --rg.inflight;
      rg.top_up(sw + 1);                                                  // refill: this sweep, then the head of the next
    }
    if (gl == gl2) {                                                      // (not the refilling thread when the group has 2+ warps)
#pragma unroll
      for (int i = 0; i < RB; ++i)
        if (i < rows) {
          ttil_s[r0 + i] = tt[i];
          sacc += (double)tt[i] * (double)tt[i];
        }
      st_release_cta(prog_s + g, rg.cons);                                // the helper warps may take these rows
    }
#pragma unroll
    for (int i = 0; i < RB; ++i)
#pragma unroll
      for (int v = 0; v < NV; ++v) axpy4(q[v], x[i][v], tt[i]);
  }
#pragma unroll
  for (int v = 0; v < NV; ++v) *reinterpret_cast<float4*>(qs + (size_t)g * ldr + 4 * (gl + GT * v)) = q[v];
  if (gl == gl2) sgrp[g] = sacc;
  cta_sync();
}

// ------------------------------------------------------------------------------------ LOADS sweep from the ring
// For every owned row r:  x = R[r,:];  (DEFL) x -= d[r]*pdef, R[r,:] = x (the pending deflation S9);
// q += x*t0[r] (S2 with the start vector).  Leaves qs[g][ldr]; ends with cta_sync().
template <int NV, int RB, bool DEFL>
__device__ __forceinline__ void sweep_loads_ring(const FusedParams& prm, Ring<RB>& rg, int sw, float* Rb,
                                                 const float* t0_s, const float* d_s, const float* pdef_s, float* qs) {
  const int GT = prm.GT, NG = kThreads / GT, ldr = prm.ldr;
  const int tid = threadIdx.x, g = tid / GT, gl = tid - g * GT;
  float4 pd[NV], q[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    pd[v] = DEFL ? *reinterpret_cast<const float4*>(pdef_s + 4 * (gl + GT * v)) : make_float4(0.f, 0.f, 0.f, 0.f);
    q[v] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  const bool rev = (sw & 1) != 0;
  for (int bq = g; bq < rg.nb; bq += NG) {
    const int bi = rev ? (rg.nb - 1 - bq) : bq;
    const int r0 = bi * RB;
    const int rows = min(RB, rg.mb - r0);
    rg.wait_next();
    const float* sl = rg.cur_slot();
    float4 x[RB][NV];
#pragma unroll
    for (int i = 0; i < RB; ++i) {
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        if (i < rows) x[i][v] = *reinterpret_cast<const float4*>(sl + (size_t)i * ldr + 4 * (gl + GT * v));
        else x[i][v] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
#pragma unroll
    for (int i = 0; i < RB; ++i) {
      if (i < rows) {
        const int r = r0 + i;
        const float dr = DEFL ? -d_s[r] : 0.f;
        const float tr = t0_s[r];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          if constexpr (DEFL) {
            axpy4(x[i][v], pd[v], dr);
            *reinterpret_cast<float4*>(Rb + (size_t)r * ldr + 4 * (gl + GT * v)) = x[i][v];
          }
          axpy4(q[v], x[i][v], tr);
        }
      }
    }
    if (GT == 32) __syncwarp();                                           // every thread of the group has read the slot
    else named_bar_sync(1 + g, GT);                                       // (its values went through the FMAs above)
    rg.consumed();
    if (gl == 0) {
      --rg.inflight;
      rg.top_up(DEFL ? sw : sw + 1);                                      // a writing sweep is not overtaken (file header)
    }
  }
#pragma unroll
  for (int v = 0; v < NV; ++v) *reinterpret_cast<float4*>(qs + (size_t)g * ldr + 4 * (gl + GT * v)) = q[v];
  if constexpr (DEFL) {
    fence_proxy_async();                                                  // my stores to R before later bulk-copy reads
    cta_sync();
    if (gl == 0) rg.top_up(sw + 1);
  }
  cta_sync();
}

// ------------------------------------------------------------------------------------ helper warps: B-partials (S6)
// hb_s[hw][j] = sum over the batches this helper warp takes of V[r, j] * t~[r]   (B = V_(k)^T t~).
// A lane owns 4 consecutive columns of a 128-column chunk (one 16-byte load per row from the row-major copy Vrm);
// the V rows of the next kHD batches are already in registers when the row group reports the batch done.
constexpr int kHD = 4;
template <int RB>
__device__ __forceinline__ void helper_main(const FusedParams& prm, int mb, long long m0, const float* ttil_s, float* hb_s,
                                            const volatile int* cmd_s, const unsigned* prog_s) {
  const int lane = threadIdx.x & 31, hw = (threadIdx.x >> 5) - kWarps;
  const int NG = kThreads / prm.GT, Kpad = prm.Kpad;
  const int nb = (mb + RB - 1) / RB;
  const int nmine = nb > hw ? (nb - hw + kHelperWarps - 1) / kHelperWarps : 0;
  const float* Vb = prm.Vrm + (size_t)m0 * Kpad;
  for (;;) {
    named_bar_sync(BAR_HSTART, kTmaThreads);
    const int cmd = cmd_s[0], k = cmd_s[1], sw = cmd_s[2];
    if (cmd == HCMD_EXIT) return;
    const bool rev = (sw & 1) != 0;
    for (int c0 = 0; c0 < k; c0 += 128) {
      const int col = c0 + 4 * lane;
      const bool active = col < k;
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
      float4 v[kHD][RB];
      auto load = [&](float4 (&dst)[RB], int i) {
        const int bq = hw + i * kHelperWarps;
        const int r0 = (rev ? (nb - 1 - bq) : bq) * RB;
#pragma unroll
        for (int r = 0; r < RB; ++r)
          dst[r] = (active && r0 + r < mb) ? __ldcg(reinterpret_cast<const float4*>(Vb + (size_t)(r0 + r) * Kpad + col))
                                           : make_float4(0.f, 0.f, 0.f, 0.f);
      };
#pragma unroll
      for (int s = 0; s < kHD; ++s)
        if (s < nmine) load(v[s], s);
      for (int i0 = 0; i0 < nmine; i0 += kHD) {
#pragma unroll
        for (int s = 0; s < kHD; ++s) {
          const int i = i0 + s;
          if (i < nmine) {
            const int bq = hw + i * kHelperWarps;
            const int gq = bq % NG;
            const unsigned need = (unsigned)sw * (unsigned)((nb - gq + NG - 1) / NG) + (unsigned)(bq / NG) + 1u;
            unsigned spins = 0;
            while ((int)(ld_acquire_cta(prog_s + gq) - need) < 0) {         // the row group has not finished this batch yet
              __nanosleep(64);                                             // (do not compete with the row groups for issue slots)
              if (++spins > (kSpinLimit << 2)) { *prm.status = 1u; break; }
            }
            const int r0 = (rev ? (nb - 1 - bq) : bq) * RB;
#pragma unroll
            for (int r = 0; r < RB; ++r) {
              if (r0 + r < mb) {
                const float t = ttil_s[r0 + r];
                acc.x = fmaf(v[s][r].x, t, acc.x);
                acc.y = fmaf(v[s][r].y, t, acc.y);
                acc.z = fmaf(v[s][r].z, t, acc.z);
                acc.w = fmaf(v[s][r].w, t, acc.w);
              }
            }
            if (i + kHD < nmine) load(v[s], i + kHD);
          }
        }
      }
      if (active) *reinterpret_cast<float4*>(hb_s + (size_t)hw * Kpad + col) = acc;
    }
    __syncwarp();
    bar_arrive(BAR_HDONE, kTmaThreads);
  }
}

// ------------------------------------------------------------------------------------ the kernel
// Launched with kTmaThreads threads: warps 0..kWarps-1 run the solve (the body below is pca_fused_kernel's streaming
// instantiation with the ring sweeps), warps kWarps.. are the B-partial helpers.
template <int NV, int RB>
__global__ void __launch_bounds__(kTmaThreads, 1) pca_tma_kernel(const FusedParams prm) {
  extern __shared__ __align__(16) unsigned char smem[];
  float* p_s = reinterpret_cast<float*>(smem + prm.off_p);        // npx: current unit loads p
  float* pdef_s = reinterpret_cast<float*>(smem + prm.off_pdef);  // ldr: loads of the previous component
  float* ttil_s = reinterpret_cast<float*>(smem + prm.off_ttil);  // Mb : t0 / t~ rows of this CTA
  float* d_s = reinterpret_cast<float*>(smem + prm.off_d);        // Mb : pending deflation vector rows
  float* qs = reinterpret_cast<float*>(smem + prm.off_qs);        // NG x ldr group partials
  float* red_s = reinterpret_cast<float*>(smem + prm.off_red);    // 2 x kWarps x RB
  double* sgrp = reinterpret_cast<double*>(smem + prm.off_sgrp);  // NG
  double* sb_s = reinterpret_cast<double*>(smem + prm.off_B);     // 4 + Kpad: |t~|^2, -, |A|^2, -, B
  double* B_s = sb_s + 4;
  double* A_s = reinterpret_cast<double*>(smem + prm.off_A);      // Kpad
  double* scr = reinterpret_cast<double*>(smem + prm.off_scr);    // kThreads
  double* ctl_s = scr + kThreads - 8;                             // lambda', decision, 1/|p^| of the current pass
  double* praw_s = reinterpret_cast<double*>(smem + prm.off_praw);// Ns: p~ / p^ slice of this owner
  float* lam_s = reinterpret_cast<float*>(smem + prm.off_lam);    // Kpad
  float* ring_s = reinterpret_cast<float*>(smem + prm.off_ring);  // NG x SG slots of RB x ldr floats
  unsigned long long* mbar_s = reinterpret_cast<unsigned long long*>(smem + prm.off_mbar);   // NG x SG
  float* hb_s = reinterpret_cast<float*>(smem + prm.off_hb);      // kHelperWarps x Kpad: helper B-partials
  volatile int* cmd_s = reinterpret_cast<volatile int*>(smem + prm.off_cmd);                // helper command
  unsigned* prog_s = reinterpret_cast<unsigned*>(smem + prm.off_prog);                      // NG progress words

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int b = blockIdx.x;
  const long long M = prm.M;
  const int N = prm.N, K = prm.K, G = prm.G, ldr = prm.ldr, Kpad = prm.Kpad, Ns = prm.Ns, Gs = prm.Gs;
  const int GT = prm.GT, NG = kThreads / GT, SG = prm.SG;
  const long long m0 = (long long)b * prm.Mb;
  const int mb = (int)max(0LL, min((long long)prm.Mb, M - m0));

  if (tid < NG * SG) mbar_init(mbar_s + tid, 1);
  if (tid < NG) prog_s[tid] = 0u;
  if (tid == 0) { cmd_s[0] = HCMD_EXIT; cmd_s[1] = 0; cmd_s[2] = 0; }
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  fence_proxy_async();
  __syncthreads();                                         // all kTmaThreads threads, once
  // register file: 20 warps = 5 per SM sub-partition = 96 registers per thread at launch; the helper warp group hands
  // registers over to the four compute warp groups (the launch holds 5 x 96 = 480 per lane slot: 4 x 104 + 64 = 480; asking for more would wait forever)
  if (w >= kWarps) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
    helper_main<RB>(prm, mb, m0, ttil_s, hb_s, cmd_s, prog_s);
    return;
  }
  asm volatile("setmaxnreg.inc.sync.aligned.u32 104;");

  const int npx = Gs * Ns;                                 // exchanged length of p (>= N)
  const int SBw = 4 + Kpad;
  const bool gs = prm.algo == 1;
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
  float* Vb = prm.Vrm + (size_t)m0 * Kpad;
  float* Pc = prm.cache_pw ? reinterpret_cast<float*>(smem + prm.off_pc) : prm.Pown + (size_t)b * Ns * Kpad;
  float* Wc = prm.cache_pw ? reinterpret_cast<float*>(smem + prm.off_wc) : prm.Wown + (size_t)b * Ns * Kpad;

  Ring<RB> rg;
  {
    const int g = tid / GT;
    rg.slots = ring_s + (size_t)g * SG * RB * ldr;
    rg.full = mbar_s + g * SG;
    rg.Rb = Rb; rg.SG = SG; rg.ldr = ldr; rg.mb = mb; rg.nb = (mb + RB - 1) / RB; rg.g = g; rg.NG = NG;
    rg.cons = 0; rg.cons_slot = 0; rg.cons_par = 0u; rg.iss_slot = 0; rg.inflight = 0; rg.iss_sw = 0; rg.iss_bq = g; rg.status = status;
    if (tid - g * GT == 0) rg.top_up(0);                   // the head of the first sweep is on its way
  }
  int sw = 0;                                              // sweeps done (loads sweeps included): row order of the next one

  for (int i = tid; i < prm.Mb; i += kThreads) d_s[i] = 0.f;
  for (int n = tid; n < max(ldr, npx); n += kThreads) {
    if (n < npx) p_s[n] = 0.f;
    if (n < ldr) pdef_s[n] = 0.f;
  }
  if (prm.cache_pw)
    for (int i = tid; i < Ns * Kpad; i += kThreads) { Pc[i] = 0.f; Wc[i] = 0.f; }
  for (int i = tid; i < Ns; i += kThreads) praw_s[i] = 0.0;
  cta_sync();

  for (int k = 0; k < K; ++k) {
    const bool gsk = gs && k > 0;
    trace_mark(prm, tn, TR_COMPONENT);
    // ---- S1: t0 <- column k of the deflated residual (reading C6) ----
    for (int i = tid; i < mb; i += kThreads) ttil_s[i] = fmaf(-d_s[i], pdef_s[k], ld_cg(Rb + (size_t)i * ldr + k));
    cta_sync();
    // ---- LOADS sweep: pending deflation (S9) + q = R^T t0 (S2) ----
    if (k == 0) sweep_loads_ring<NV, RB, false>(prm, rg, sw, Rb, ttil_s, d_s, pdef_s, qs);
    else        sweep_loads_ring<NV, RB, true>(prm, rg, sw, Rb, ttil_s, d_s, pdef_s, qs);
    ++sw;
    ++seq;
    {
      const unsigned par = seq & 1u;
      publish_q_ll(prm, qs, prm.Qx + (size_t)par * Gs * G * Ns, b, seq);
      double s = 0.0;
      for (int i = tid; i < mb; i += kThreads) { const double v = (double)ttil_s[i]; s += v * v; }
      s = block_sum_c(s, scr);
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
      hop_wait_c(cnt1, e1, status);
      {
        LLJob jq, jsb;
        jq.base = prm.Qx + ((size_t)par * Gs + b) * G * Ns; jq.out = praw_s; jq.units = owner ? (Ns >> 1) : 0;
        jq.nparts = G; jq.stride = Ns; jq.f64_unit0 = false;
        jsb.base = prm.SBx + (size_t)par * G * SBw; jsb.out = sb_s; jsb.units = (gsk && !first) ? 2 + ((k + 1) >> 1) : 1;
        jsb.nparts = G; jsb.stride = SBw; jsb.f64_unit0 = 2;
        if (jsb.units <= 16) {
          ll_reduce2(jsb, jq, seq, status);
        } else {
          RegGather gsb;
          int hs = 32;
          while (hs < jsb.units) hs <<= 1;
          gsb.base = jsb.base; gsb.stride = SBw; gsb.hp = hs; gsb.npairs = jsb.units; gsb.nparts = G; gsb.f64_pair0 = 2;
          gsb.red = reinterpret_cast<double2*>(qs); gsb.out = sb_s;
          u64 sx[8], sy[8];
          reg_gather_issue<8>(gsb, sx, sy);
          jsb.units = 0;
          ll_reduce2(jsb, jq, seq, status);
          reg_gather_finish<8>(gsb, sx, sy, seq, status);
          cta_sync();
          reg_gather_store(gsb);
        }
      }
      cta_sync();
      trace_mark(prm, tn, TR_X1);
      // S7/S8 by warp 0; meanwhile the owners' other warps start on p~ = q - W B
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
            // S8: listings' strict relative test (reading C3) (+ reading C4b)
            if (pca_stagnated(lam, lam2, ln, prm.eps, prm.test_mode, prm.stag2) || (it >= prm.max_iter)) st = 1;
          }
        }
        if (lane == 0) { ctl_s[0] = ln; reinterpret_cast<int*>(ctl_s + 1)[0] = st; }
      }
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
      cta_sync();
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
        hop_wait_c(cnt2, e2, status);
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
          cta_sync();
          reg_gather_store(ga);
        }
        cta_sync();
        trace_mark(prm, tn, TR_X2);
        slice_correct(praw_s, Pc, A_s, ns, k, Kpad);
        cta_sync();
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
          hop_arrive(cnt3);
        }
      }
      trace_mark(prm, tn, TR_PHAT);
      e3 += (unsigned)Gs;
      hop_wait_c(cnt3, e3, status);
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
      cta_sync();
      trace_mark(prm, tn, TR_X3);
      inv_pn = reinterpret_cast<const float*>(ctl_s + 1)[1];                  // p = p~/|p~| (see S3 above)
      const double a2mine = gsk ? scr[4] : 0.0;
      if (!(inv_pn > 0.f)) { degenerate = true; break; }                      // reading C7
      for (int n = tid; n < npx; n += kThreads) p_s[n] *= inv_pn;             // each thread rescales what it wrote
      if (gsk && tid == 0) { cmd_s[0] = HCMD_SWEEP; cmd_s[1] = k; cmd_s[2] = sw; }
      cta_sync();
      first = false;
      trace_mark(prm, tn, TR_PREADY);
      // ---- FUSED sweep: t~ = R p (S5), q = R^T t~, s = |t~|^2; helper warps: B-partials V^T t~ (S6) ----
      ++seq;
      ++it;
      {
        const unsigned npar = seq & 1u;
        if (gsk) bar_arrive(BAR_HSTART, kTmaThreads);                         // the helpers start following the row groups
        sweep_fused_ring<NV, RB>(prm, rg, sw, p_s, ttil_s, qs, red_s, sgrp, prog_s);
        ++sw;
        trace_mark(prm, tn, TR_SWEEP);
        publish_q_ll(prm, qs, prm.Qx + (size_t)npar * Gs * G * Ns, b, seq);
        u64* sbx = prm.SBx + ((size_t)npar * G + b) * SBw;
        if (tid == 0) {
          double a = 0.0;
          for (int g = 0; g < NG; ++g) a += sgrp[g];
          ll_st2d(sbx, a, seq);
          if (gsk) ll_st2d(sbx + 2, a2mine, seq);
        }
        if (gsk) {
          named_bar_sync(BAR_HDONE, kTmaThreads);                             // the helpers' partial sums are in hb_s
          for (int j0 = 2 * tid; j0 < k; j0 += 2 * kThreads) {
            float s0 = 0.f, s1 = 0.f;
#pragma unroll
            for (int h = 0; h < kHelperWarps; ++h) {
              s0 += hb_s[(size_t)h * Kpad + j0];
              if (j0 + 1 < k) s1 += hb_s[(size_t)h * Kpad + j0 + 1];
            }
            ll_st2(sbx + 4 + j0, ll_wordf(s0, seq), ll_wordf(s1, seq));
          }
        }
        cta_sync();                                                           // all LL stores of this CTA are issued
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
          cta_sync();
          reg_gather_store(ga);
        }
        cta_sync();
        for (int i = tid; i < Ns; i += kThreads) praw2_s[i] = (i < ns) ? (double)p_s[n0 + i] : 0.0;
        for (int j = tid; j < k; j += kThreads) A_s[j] *= (double)inv_pn;   // A of the scaled vector p~/|p~|
        cta_sync();
        slice_correct(praw2_s, Pc, A_s, ns, k, Kpad);
        cta_sync();
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
      hop_wait_c(cnt4, e4, status);
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
      cta_sync();
      const float inv_f = reinterpret_cast<const float*>(ctl_s + 1)[1];
      for (int n = tid; n < npx; n += kThreads) p_s[n] *= inv_f;
      cta_sync();
    }
    // ---- component done ----
    if (degenerate) {
      for (int i = tid; i < mb; i += kThreads) {
        Tb[(size_t)k * M + i] = 0.f; d_s[i] = 0.f;
        if (gs) Vb[(size_t)i * Kpad + k] = 0.f;
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
        if (gs) Vb[(size_t)i * Kpad + k] = t * inv;                           // row-major copy for the helper warps
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
    cta_sync();
    trace_mark(prm, tn, TR_FINAL);
  }
  if (prm.trace_cap > 0 && b == 0 && tid == 0) prm.trace[0] = (unsigned long long)tn;

  // release the helper warps and drain the ring: no bulk copy may be in flight when the CTA exits
  if (tid == 0) cmd_s[0] = HCMD_EXIT;
  bar_arrive(BAR_HSTART, kTmaThreads);
  if (tid == rg.g * GT) {                                  // (only the group leaders know how many copies they issued)
    while (rg.inflight > 0) {
      rg.wait_next();
      rg.consumed();
      --rg.inflight;
    }
  }
  // ---- S10: GS-PCA  T <- V Lambda; skipped for the SVD output V, U, Lambda ----
  if (gs && !prm.out_svd) {
    cta_sync();
    for (int kk = 0; kk < K; ++kk) {
      const float l = lam_s[kk];
      for (int i = tid; i < mb; i += kThreads) Tb[(size_t)kk * M + i] *= l;
    }
  }
}

}  // namespace pca
