// =====================================================================================
// pca_api.cu -- host side of the C ABI declared in include/pca.h: argument checks, the launch
// plan (path, CTAs, lane mapping, shared-memory carve-up, workspace layout) and the launches.
// No torch types, no exceptions across the boundary, no printing.
// =====================================================================================
#include "../../include/pca.h"

#include <cuda_runtime.h>

#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <new>

#include "pca_center.cuh"
#include "pca_fused.cuh"
#include "pca_one.cuh"
#include "pca_reg.cuh"
#include "pca_solve.cuh"
#include "pca_tma.cuh"

using pca::FusedParams;
using pca::RegParams;
using pca::OneParams;
using pca::SolveParams;

namespace {

inline long long round_up(long long v, long long a) { return (v + a - 1) / a * a; }
inline long long ceil_div(long long a, long long b) { return (a + b - 1) / b; }

typedef void (*solve_kernel_t)(const SolveParams);

struct Variant { int resident, vec, tr, rc; solve_kernel_t fn; };

#define PCA_VARIANT(RES, VEC, TR, RC) {RES, VEC, TR, RC, pca::pca_solve_kernel<(RES != 0), VEC, TR, RC>}
const Variant kVariants[] = {
    PCA_VARIANT(0, 4, 32, 1), PCA_VARIANT(0, 4, 32, 2), PCA_VARIANT(0, 4, 32, 4),
    PCA_VARIANT(0, 4, 8, 1),  PCA_VARIANT(0, 4, 8, 2),  PCA_VARIANT(0, 4, 8, 4),
    PCA_VARIANT(0, 1, 32, 4),
    PCA_VARIANT(1, 4, 32, 1), PCA_VARIANT(1, 4, 32, 2), PCA_VARIANT(1, 4, 32, 4),
    PCA_VARIANT(1, 4, 8, 1),  PCA_VARIANT(1, 4, 8, 2),  PCA_VARIANT(1, 4, 8, 4),
    PCA_VARIANT(1, 1, 32, 4),
};
#undef PCA_VARIANT

typedef void (*fused_kernel_t)(const FusedParams);
struct FusedVariant { int resident, nv; fused_kernel_t fn; };
#define PCA_FVARIANT(RES, NV) {RES, NV, pca::pca_fused_kernel<NV, (RES != 0)>}
const FusedVariant kFusedVariants[] = {
    PCA_FVARIANT(0, 1), PCA_FVARIANT(0, 2), PCA_FVARIANT(0, 3), PCA_FVARIANT(0, 4),
    PCA_FVARIANT(1, 1), PCA_FVARIANT(1, 2), PCA_FVARIANT(1, 3), PCA_FVARIANT(1, 4),
};
#undef PCA_FVARIANT

// TMA-staged streaming kernel (pca_tma.cuh): NV float4 per thread per row, RB rows per ring slot
struct TmaVariant { int nv, rb; fused_kernel_t fn; };
#define PCA_TVARIANT(NV, RB) {NV, RB, pca::pca_tma_kernel<NV, RB>}
const TmaVariant kTmaVariants[] = {
    PCA_TVARIANT(1, 2), PCA_TVARIANT(2, 2), PCA_TVARIANT(3, 2), PCA_TVARIANT(4, 2), PCA_TVARIANT(4, 1), PCA_TVARIANT(4, 4),
};
#undef PCA_TVARIANT

}  // namespace

namespace pca {
reg_kernel_t reg_kernel_lookup_part0(int gt, int rpt);
reg_kernel_t reg_kernel_lookup_part1(int gt, int rpt);
reg_kernel_t reg_kernel_lookup_part2(int gt, int rpt);
reg_kernel_t reg_kernel_lookup_part3(int gt, int rpt);
reg_kernel_t reg_kernel_lookup_part4(int gt);
reg_kernel_t reg_kernel_lookup_part5(int gt);
one_kernel_t one_kernel_lookup_part0(int gt, int rpt);
one_kernel_t one_kernel_lookup_part1(int gt, int rpt);
one_kernel_t one_kernel_lookup(int gt, int rpt) {
  one_kernel_t f = one_kernel_lookup_part0(gt, rpt);
  if (!f) f = one_kernel_lookup_part1(gt, rpt);
  return f;
}
reg_kernel_t reg_kernel_lookup(int gt, int rpt, int rs) {
  if (rs != 0) {
    if (rs != kRegSmemRows || rpt != 7) return nullptr;
    reg_kernel_t g = reg_kernel_lookup_part4(gt);
    return g ? g : reg_kernel_lookup_part5(gt);
  }
  reg_kernel_t f = reg_kernel_lookup_part0(gt, rpt);
  if (!f) f = reg_kernel_lookup_part1(gt, rpt);
  if (!f) f = reg_kernel_lookup_part2(gt, rpt);
  if (!f) f = reg_kernel_lookup_part3(gt, rpt);
  return f;
}
}  // namespace pca

struct pca_ctx {
  long long M = 0, N = 0;
  int K = 0;
  double eps = 0;
  int max_iter = 0;
  int algo = 0;
  // device
  int device = 0, num_sms = 0, smem_optin = 0;
  // options
  int opt_path = 0, opt_ctas = 0, opt_center_mode = 0, opt_trace = 0, opt_owners = 0, opt_kdirect = -1, opt_test_mode = 0;
  int opt_stag2 = 1, opt_output = 0, opt_gs_passes = 1, opt_ring_rows = 0, opt_ring_slots = 0, opt_storage = 0, opt_defer_s3 = 1;
  // plan
  bool planned = false;
  int path = 0;  // 1 streaming, 2 resident (two-sweep kernel); 3 streaming, 4 resident (single-sweep kernel);
                 // 5 register-resident single-sweep kernel
  pca::reg_kernel_t rfn = nullptr;
  RegParams rprm{};
  pca::one_kernel_t ofn = nullptr;   // path 6: one-CTA kernel
  OneParams oprm{};
  int r_gt = 0, r_rpt = 0;
  size_t ws_off_bx = 0;
  const Variant* variant = nullptr;
  SolveParams prm{};
  pca::SolveParamsT<double> prm64{};   // PCA_OPT_STORAGE = 1
  const FusedVariant* fvariant = nullptr;
  fused_kernel_t ffn = nullptr;      // the kernel of paths 3, 4, 7
  int ring_rows = 0;
  size_t ws_off_vrm = 0, ws_off_pfx = 0, ws_off_nfx = 0;
  FusedParams fprm{};
  size_t ws_off_rrm = 0, ws_off_xchg = 0, ws_xchg_bytes = 0, ws_off_qx = 0, ws_off_sbx = 0, ws_off_ax = 0, ws_off_px = 0,
         ws_off_nx = 0, ws_off_pown = 0, ws_off_wown = 0, ws_off_status = 0, ws_off_cnt = 0, ws_off_trace = 0;
  size_t smem_bytes = 0;
  size_t ws_bytes = 0;
  size_t ws_off_ppart = 0, ws_off_apart = 0, ws_off_bpart = 0, ws_off_pvec = 0, ws_off_qpart = 0, ws_off_spart = 0,
         ws_off_bar = 0;
  // workspace (caller-owned)
  void* ws = nullptr;
  size_t ws_given = 0;
  bool ran = false;
  // private staging for pca_fit_host
  float *hX = nullptr, *hT = nullptr, *hP = nullptr, *hLam = nullptr;
  int* hIters = nullptr;
  void* hWs = nullptr;
  size_t hWs_bytes = 0;
  int last_cuda = 0;
};

namespace {

int cuda_fail(pca_ctx* c, cudaError_t e) {
  c->last_cuda = (int)e;
  return PCA_ECUDA;
}
#define PCA_CUDA(c, expr)                                \
  do {                                                   \
    cudaError_t e__ = (expr);                            \
    if (e__ != cudaSuccess) return cuda_fail((c), e__);  \
  } while (0)

const Variant* find_variant(int resident, int vec, int tr, int rc) {
  for (const Variant& v : kVariants)
    if (v.resident == resident && v.vec == vec && v.tr == tr && v.rc == rc) return &v;
  return nullptr;
}

// Lane mapping for a slab of `rv` row-vectors per column: smallest TR*RC >= rv (ties: wider TR),
// else the largest mapping with a row-chunk loop.
void choose_mapping(int vec, long long rv, int* tr, int* rc) {
  if (vec == 1) { *tr = 32; *rc = 4; return; }
  const int cand[6][2] = {{32, 1}, {32, 2}, {32, 4}, {8, 1}, {8, 2}, {8, 4}};
  int best = -1;
  long long best_cap = 0;
  for (int i = 0; i < 6; ++i) {
    const long long cap = (long long)cand[i][0] * cand[i][1];
    if (cap >= rv && (best < 0 || cap < best_cap)) { best = i; best_cap = cap; }
  }
  if (best < 0) { *tr = 32; *rc = 4; return; }
  *tr = cand[best][0];
  *rc = cand[best][1];
}

// Fill prm's geometry + shared-memory carve-up for a given (path, G).  Returns dynamic smem bytes.
size_t carve(pca_ctx* c, int resident, int G, int vec, SolveParams* p, int* tr, int* rc, size_t esz = 4) {
  const long long M = c->M, N = c->N;
  p->G = G;
  p->Mb = (int)round_up(ceil_div(M, G), vec);
  p->Ns = (int)round_up(ceil_div(N, G), 4);
  p->Gs = (int)ceil_div(N, p->Ns);
  p->Npad = (int)round_up(N, 4);
  p->Kpad = (int)round_up(c->K, 4);
  p->slab_ld = resident ? (int)round_up(p->Mb, 4) : 0;
  choose_mapping(vec, ceil_div(p->Mb, vec), tr, rc);
  const int ch = vec * (*tr) * (*rc);
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = (size_t)round_up((long long)(off + bytes), 16); return (int)o; };
  p->off_t = take((size_t)round_up(p->Mb, 4) * esz);
  p->off_d = take((size_t)round_up(p->Mb, 4) * esz);
  p->off_p = take((size_t)p->Npad * esz);
  p->off_slice = take((size_t)p->Ns * esz);
  p->off_coef = take((size_t)p->Kpad * 8);
  p->off_lam = take((size_t)p->Kpad * esz);
  p->off_scr = take((size_t)pca::kThreads * 8);
  p->off_red = take((size_t)pca::kWarps * ch * esz);
  p->off_slab = take(resident ? (size_t)p->slab_ld * (size_t)N * esz : 0);
  return off;
}

// Single-sweep kernel (pca_fused.cuh): GT threads share a row, NV float4 per thread per row.
// want: 0 = resident if it fits else streaming, 3 = streaming, 4 = resident.
int make_fused_plan(pca_ctx* c, int want) {
  const long long M = c->M, N = c->N;
  const int sms = c->num_sms;
  int GT = 32;
  while ((long long)16 * GT < N) GT *= 2;
  if (GT > pca::kThreads) return PCA_EUNSUPPORTED;
  // the k-vectors A and B are combined with one thread per pair of entries (RegGather): at most kThreads pairs.
  // Larger K with GS-PCA goes to the two-sweep kernel, whose coefficient reduction is chunked.
  if (c->algo == PCA_ALGO_GS && (c->K + 1) / 2 + 1 > pca::kThreads) return PCA_EUNSUPPORTED;
  const int NV = (int)ceil_div(N, 4LL * GT);
  const int ldr = 4 * GT * NV;
  const int g_min = (int)ceil_div(N, pca::kThreads);
  int tma_rb = 0;                                                     // > 0: TMA plan with tma_rb rows per ring slot
  bool tma_no_cache = false;
  auto carve_fused = [&](int resident, int G, FusedParams* p) -> size_t {
    p->G = G;
    p->Mb = (int)ceil_div(M, G);
    p->ldr = ldr; p->GT = GT;
    p->Ns = (int)round_up(ceil_div(N, G), 4);
    p->Gs = (int)ceil_div(N, p->Ns);
    p->Kpad = (int)round_up(c->K, 4);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = (size_t)round_up((long long)(off + bytes), 16); return (int)o; };
    const size_t mbp = (size_t)round_up(p->Mb, 4);
    const size_t npx = (size_t)p->Gs * p->Ns;
    p->off_p = take((npx > (size_t)ldr ? npx : (size_t)ldr) * 4);
    p->off_pdef = take((size_t)ldr * 4);
    p->off_ttil = take(mbp * 4);
    p->off_d = take(mbp * 4);
    p->off_qs = take((size_t)pca::kThreads * 4 * NV * 4);
    p->off_red = take((size_t)2 * pca::kWarps * pca::kRB * 4);
    p->off_sgrp = take((size_t)(pca::kThreads / GT) * 8);
    p->off_B = take((size_t)(4 + p->Kpad) * 8);
    p->off_A = take((size_t)p->Kpad * 8);
    p->off_scr = take((size_t)pca::kThreads * 8);
    p->off_praw = take((size_t)2 * p->Ns * 8);
    p->off_lam = take((size_t)p->Kpad * 4);
    // owner-private panels P[slice, :], W[slice, :]: shared memory unless that crowds out the rest
    const size_t panel = (size_t)p->Ns * p->Kpad * 4;
    const size_t slab_bytes = resident ? (size_t)p->Mb * (size_t)ldr * 4 : 0;
    p->cache_pw = (off + 2 * panel + slab_bytes <= (size_t)c->smem_optin && 2 * panel <= (size_t)64 * 1024) ? 1 : 0;
    if (tma_rb && (tma_no_cache || 2 * panel > (size_t)32 * 1024)) p->cache_pw = 0;
    p->off_pc = take(p->cache_pw ? panel : 0);
    p->off_wc = take(p->cache_pw ? panel : 0);
    p->off_slab = take(resident ? (size_t)p->Mb * (size_t)ldr * 4 : 0);
    // what is left of the shared memory caches the CTA's rows of the first Ksm unit score vectors (GS-PCA, B-partials S6)
    p->Mbp = (int)round_up(p->Mb, 32);
    p->Ksm = 0;
    p->off_vc = (int)off;
    p->SG = 0;
    if (tma_rb) {
      // ring: NG groups x SG slots of tma_rb rows; everything that is left of the shared memory, at most 8 slots per group
      p->off_hb = take((size_t)pca::kHelperWarps * p->Kpad * 4);
      p->off_cmd = take(16);
      p->off_prog = take((size_t)(pca::kThreads / GT) * 4);
      const int NG = pca::kThreads / GT;
      p->off_mbar = take((size_t)NG * 8 * 8);
      off = (size_t)round_up((long long)off, 128);
      const size_t slot = (size_t)tma_rb * ldr * 4;
      long long sg = ((long long)c->smem_optin - (long long)off) / (long long)(slot * NG);
      const long long need = ceil_div(ceil_div(p->Mb, tma_rb), NG);        // batches per group and sweep
      if (sg > 8) sg = 8;
      if (sg > need + 1) sg = need + 1;
      if (c->opt_ring_slots > 0 && sg > c->opt_ring_slots) sg = c->opt_ring_slots;
      if (sg < 1) return (size_t)c->smem_optin + 1;                         // does not fit
      p->SG = (int)sg;
      p->off_ring = take((size_t)NG * sg * slot);
      return off;
    }
    // (streaming plan: not beyond 100 KB in total -- the sweep keeps 128 KB of loads in flight per SM and those need L1 lines;
    //  measured on config 4: with all 227 KB as shared memory the sweep is 33 % slower)
    const long long cap = resident ? (long long)c->smem_optin : (100LL * 1024 < c->smem_optin ? 100LL * 1024 : (long long)c->smem_optin);
    if (c->algo == PCA_ALGO_GS && (long long)off + 4096 < cap) {
      long long ks = (cap - (long long)off - 1024) / ((long long)p->Mbp * 4);
      if (ks > c->K) ks = c->K;
      ks &= ~1LL;                                                     // pairs of columns
      if (ks > 0) { p->Ksm = (int)ks; p->off_vc = take((size_t)ks * p->Mbp * 4); }
    }
    return off;
  };
  auto find = [&](int resident) -> const FusedVariant* {
    for (const FusedVariant& v : kFusedVariants)
      if (v.resident == resident && v.nv == NV) return &v;
    return nullptr;
  };
  FusedParams p{};
  size_t smem = 0;
  int path = 0;
  const FusedVariant* var = nullptr;
  auto try_plan = [&](int resident, int G) -> bool {
    if (G < g_min) G = g_min;
    if (G > sms) G = sms;
    if (G < 1) G = 1;
    if (g_min > sms) return false;
    smem = carve_fused(resident, G, &p);
    if (smem > (size_t)c->smem_optin) return false;
    var = find(resident);
    return var != nullptr;
  };
  bool ok = false;
  const TmaVariant* tvar = nullptr;
  if (want == 7) {
    const int G = c->opt_ctas > 0 ? c->opt_ctas : sms;
    const int prefer[3] = {c->opt_ring_rows > 0 ? c->opt_ring_rows : 2, 1, 4};
    for (int pi = 0; pi < (c->opt_ring_rows > 0 ? 1 : 3) && !ok; ++pi)
      for (int nc = 0; nc < 2 && !ok; ++nc) {
        tma_rb = prefer[pi];
        tma_no_cache = nc == 1;
        tvar = nullptr;
        for (const TmaVariant& v : kTmaVariants)
          if (v.nv == NV && v.rb == tma_rb) tvar = &v;
        if (!tvar) continue;
        int Gc = G < g_min ? g_min : G;
        if (Gc > sms || g_min > sms) continue;
        smem = carve_fused(0, Gc, &p);
        if (smem <= (size_t)c->smem_optin && (p.SG >= 2 || (pi == 2 && nc == 1) || c->opt_ring_rows > 0)) ok = true;
      }
    if (!ok) return PCA_EUNSUPPORTED;
    path = 7;
  }
  if (!ok && (want == 0 || want == 4)) {
    int G = c->opt_ctas > 0 ? c->opt_ctas : ((size_t)M * (size_t)ldr * 4 <= (size_t)160 * 1024 ? 1 : sms);
    ok = try_plan(1, G);
    if (!ok && c->opt_ctas == 0 && G != sms) ok = try_plan(1, sms);
    if (ok) path = 4;
    else if (want == 4) return PCA_EUNSUPPORTED;
  }
  if (!ok) {
    ok = try_plan(0, c->opt_ctas > 0 ? c->opt_ctas : sms);
    if (!ok) return PCA_EUNSUPPORTED;
    path = 3;
  }
  fused_kernel_t fn = path == 7 ? tvar->fn : var->fn;
  const int nthreads = path == 7 ? pca::kTmaThreads : pca::kThreads;
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin);   // per FUNCTION: the device maximum, so that contexts do not lower it for each other
  if (e != cudaSuccess) return cuda_fail(c, e);
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, nthreads, smem);
  if (e != cudaSuccess) return cuda_fail(c, e);
  if ((long long)per_sm * sms < p.G) return PCA_EUNSUPPORTED;

  p.M = M; p.N = (int)N; p.K = c->K; p.eps = c->eps; p.max_iter = c->max_iter; p.algo = c->algo; p.test_mode = c->opt_test_mode; p.stag2 = c->opt_stag2; p.out_svd = c->opt_output; p.defer_s3 = c->opt_defer_s3;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = (size_t)round_up((long long)(off + bytes), 256); return o; };
  take((size_t)M * (size_t)N * 4);                                   // residual of eq. (4), column-major (ABI layout)
  c->ws_off_rrm = take((size_t)M * (size_t)ldr * 4);                 // working residual, row-major
  // LL exchange buffers + status word: one contiguous region, zeroed before every launch
  c->ws_off_xchg = off;
  c->ws_off_qx = take((size_t)2 * p.Gs * p.G * p.Ns * 8);
  c->ws_off_sbx = take((size_t)2 * p.G * (4 + p.Kpad) * 8);
  c->ws_off_ax = take((size_t)2 * p.Gs * p.Kpad * 8);
  c->ws_off_px = take((size_t)2 * p.Gs * p.Ns * 8);
  c->ws_off_nx = take((size_t)2 * p.Gs * 2 * 8);
  c->ws_off_pfx = take((size_t)2 * p.Gs * p.Ns * 8);
  c->ws_off_nfx = take((size_t)2 * p.Gs * 2 * 8);
  c->ws_off_pown = take(p.cache_pw ? 0 : (size_t)p.Gs * p.Ns * p.Kpad * 4);
  c->ws_off_wown = take(p.cache_pw ? 0 : (size_t)p.Gs * p.Ns * p.Kpad * 4);
  c->ws_off_status = take(256);
  c->ws_off_cnt = take(1024);
  c->ws_xchg_bytes = off - c->ws_off_xchg;
  c->ws_off_trace = take(c->opt_trace > 0 ? ((size_t)c->opt_trace + 1 + 2 * p.G) * 8 : 0);   // records, then per-CTA sweep cycles and SM ids
  c->ws_off_vrm = take(path == 7 && c->algo == PCA_ALGO_GS ? (size_t)M * p.Kpad * 4 : 0);
  p.trace_cap = c->opt_trace;
  c->ws_bytes = off;
  c->fprm = p;
  c->fvariant = var;
  c->ffn = fn;
  c->ring_rows = tma_rb;
  c->smem_bytes = smem;
  c->path = path;
  c->planned = true;
  c->ws = nullptr;
  c->ws_given = 0;
  c->ran = false;
  return PCA_OK;
}

// Register-resident single-sweep kernel (pca_reg.cuh): GT threads share a row, 8 columns per thread, RPT rows per
// row group, the whole row block of a CTA in registers.  Fits when ceil(M/G) <= (512/GT)*7 with G <= #SMs.
int make_reg_plan(pca_ctx* c) {
  const long long M = c->M, N = c->N;
  const int sms = c->num_sms;
  int GT = 8;
  while (8LL * GT < N) GT *= 2;
  if (GT > pca::kThreads) return PCA_EUNSUPPORTED;
  if (c->algo == PCA_ALGO_GS && (c->K + 1) / 2 + 1 > pca::kThreads) return PCA_EUNSUPPORTED;   // as make_fused_plan
  const int NG = pca::kThreads / GT, ldr = 8 * GT;
  int G = c->opt_ctas > 0 ? c->opt_ctas : (int)ceil_div(M, (long long)NG * 7);
  if (G < 1) G = 1;
  if (G > sms) return PCA_EUNSUPPORTED;
  const int Mb = (int)ceil_div(M, G);
  int RPT = 0;
  for (int r : {2, 4, 7})
    if ((long long)NG * r >= Mb) { RPT = r; break; }
  if (!RPT) return PCA_EUNSUPPORTED;
  pca::reg_kernel_t fn = pca::reg_kernel_lookup(GT, RPT, 0);
  if (!fn) return PCA_EUNSUPPORTED;
  int rsm_rows = 0;                                                  // rows of every thread's row block kept in shared memory
  int g2 = 1;
  while (g2 * 2 <= G) g2 *= 2;                                       // owners: a power of two <= G
  RegParams p{};
  p.G = G; p.Mb = Mb; p.ldr = ldr; p.Kpad = (int)round_up(c->K, 4);
  const bool gs = c->algo == PCA_ALGO_GS;
  size_t smem = 0;
  auto carve_reg = [&](int Gs) -> size_t {
    p.Gs = Gs; p.Ns = ldr / Gs;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = (size_t)round_up((long long)(off + bytes), 16); return (int)o; };
    const size_t rows = (size_t)NG * RPT;
    p.off_p = take((size_t)2 * ldr * 4);
    p.off_ttil = take(rows * 4);
    p.off_d = take(rows * 4);
    p.off_qs = take((size_t)NG * ldr * 4);
    p.off_red = take((size_t)pca::kThreads * 4);
    p.off_sgrp = take((size_t)NG * 8);
    p.off_B = take((size_t)(4 + p.Kpad) * 8);
    p.off_A = take((size_t)(2 + p.Kpad) * 8);
    p.off_scr = take((size_t)pca::kThreads * 8);
    p.off_praw = take((size_t)2 * p.Ns * 8);
    const size_t KV = (size_t)(p.Kpad | 1);                           // odd row stride (bank-conflict-free both ways)
    p.off_vb = take(gs ? rows * KV * 4 : 0);
    p.off_pc = take(gs ? (size_t)p.Ns * KV * 4 : 0);
    p.off_wc = take(gs ? (size_t)p.Ns * KV * 4 : 0);
    p.off_rsm = take((size_t)rsm_rows * NG * ldr * 4);               // RowBlock: rows kept in shared memory
    p.off_x = -1;
    if (G == 1) {                                                     // one CTA: exchange buffers in shared memory if they fit
      const size_t xwords = (size_t)6 * ldr + 4 * (1 + p.Kpad / 2) + 4 * (2 + p.Kpad) + 4 * (p.Kpad / 2) + 2 * (Gs * 2 + 6) + 2 * (Gs * 2);
      if (off + xwords * 8 <= (size_t)c->smem_optin) p.off_x = take(xwords * 8);
    }
    return off;
  };
  int Gs = c->opt_owners > 0 ? c->opt_owners : 32;
  if (Gs > g2) Gs = g2;
  if (Gs > ldr / 2) Gs = ldr / 2;
  int gq = 1;
  while (gq * 2 <= Gs) gq *= 2;
  Gs = gq;
  for (;;) {
    smem = carve_reg(Gs);
    if (smem <= (size_t)c->smem_optin) break;
    if (Gs * 2 > g2 || Gs * 2 > ldr / 2) return PCA_EUNSUPPORTED;   // more owners = smaller P / W panels per owner
    Gs *= 2;
  }
  // RPT = 7 fills the register file (56 of 128 registers hold R, the rest of the pass spills): take the variant that keeps two
  // of the seven rows in shared memory when that leaves the total at or below 100 KB -- beyond it the L1 that serves the
  // remaining spills and the panel loads shrinks and the pass gets slower (measured: config 2 9.7 -> 9.3 us, config 5 with its
  // 115 KB of unit scores 11.9 -> 13.1)
  if (RPT == 7) {
    pca::reg_kernel_t fs = pca::reg_kernel_lookup(GT, RPT, pca::kRegSmemRows);
    rsm_rows = pca::kRegSmemRows;
    const size_t smem_s = carve_reg(Gs);
    if (fs && smem_s <= (size_t)100 * 1024) { fn = fs; smem = smem_s; }
    else { rsm_rows = 0; smem = carve_reg(Gs); }
  }
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin);   // per FUNCTION: the device maximum, so that contexts do not lower it for each other
  if (e != cudaSuccess) return cuda_fail(c, e);
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, pca::kThreads, smem);
  if (e != cudaSuccess) return cuda_fail(c, e);
  if ((long long)per_sm * sms < G) return PCA_EUNSUPPORTED;

  p.M = M; p.N = (int)N; p.K = c->K; p.eps = c->eps; p.max_iter = c->max_iter; p.algo = c->algo; p.test_mode = c->opt_test_mode; p.stag2 = c->opt_stag2; p.out_svd = c->opt_output; p.defer_s3 = c->opt_defer_s3;
  p.kdirect = c->opt_kdirect >= 0 ? (c->opt_kdirect > 30 ? 30 : c->opt_kdirect) : 0;    // direct: <= 16 units, one per warp
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = (size_t)round_up((long long)(off + bytes), 256); return o; };
  take((size_t)M * (size_t)N * 4);                                   // residual of eq. (4), column-major (ABI layout)
  c->ws_off_rrm = take((size_t)M * (size_t)ldr * 4);                 // row-major copy: read once, written once
  c->ws_off_xchg = off;
  c->ws_off_qx = take((size_t)2 * G * ldr * 8);
  c->ws_off_sbx = take((size_t)2 * G * (2 + p.Kpad) * 8);
  c->ws_off_bx = take((size_t)2 * (2 + p.Kpad) * 2 * 8);
  c->ws_off_ax = take((size_t)2 * p.Gs * p.Kpad * 8);
  c->ws_off_px = take((size_t)2 * ldr * 8);
  c->ws_off_nx = take((size_t)2 * (p.Gs * 2 + 6) * 8);
  c->ws_off_pfx = take((size_t)2 * ldr * 8);
  c->ws_off_nfx = take((size_t)2 * p.Gs * 2 * 8);
  c->ws_off_status = take(256);
  c->ws_xchg_bytes = off - c->ws_off_xchg;
  c->ws_off_trace = take(c->opt_trace > 0 ? ((size_t)c->opt_trace + 1) * 8 : 0);
  p.trace_cap = c->opt_trace;
  c->ws_bytes = off;
  c->rprm = p;
  c->rfn = fn;
  c->r_gt = GT; c->r_rpt = RPT;
  c->smem_bytes = smem;
  c->path = 5;
  c->planned = true;
  c->ws = nullptr;
  c->ws_given = 0;
  c->ran = false;
  return PCA_OK;
}

// One-CTA kernel (pca_one.cuh): the whole matrix in the registers of one SM.  M <= (512/GT)*7, GT = pow2 >= N/8, GT <= 64.
int make_one_plan(pca_ctx* c) {
  const long long M = c->M, N = c->N;
  int GT = 8;
  while (8LL * GT < N) GT *= 2;
  if (GT > 64) return PCA_EUNSUPPORTED;
  const int NG = pca::kThreads / GT, ldr = 8 * GT;
  if (M > (long long)NG * 7 || (c->opt_ctas > 1)) return PCA_EUNSUPPORTED;
  int RPT = 0;
  for (int r : {2, 4, 7})
    if ((long long)NG * r >= M) { RPT = r; break; }
  pca::one_kernel_t fn = pca::one_kernel_lookup(GT, RPT);
  if (!fn) return PCA_EUNSUPPORTED;
  OneParams p{};
  p.M = (int)M; p.N = (int)N; p.K = c->K; p.eps = c->eps; p.max_iter = c->max_iter; p.algo = c->algo; p.test_mode = c->opt_test_mode; p.stag2 = c->opt_stag2; p.out_svd = c->opt_output;
  p.ldr = ldr; p.Kpad = (int)round_up(c->K, 4);
  const bool gs = c->algo == PCA_ALGO_GS;
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
  if (smem > (size_t)c->smem_optin) return PCA_EUNSUPPORTED;
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin);   // per FUNCTION: the device maximum, so that contexts do not lower it for each other
  if (e != cudaSuccess) return cuda_fail(c, e);
  size_t woff = 0;
  auto wtake = [&](size_t bytes) { size_t o = woff; woff = (size_t)round_up((long long)(woff + bytes), 256); return o; };
  wtake((size_t)M * (size_t)N * 4);                                  // residual of eq. (4), column-major (ABI layout)
  c->ws_off_rrm = wtake((size_t)M * (size_t)ldr * 4);                // row-major copy: read once, written once
  c->ws_off_status = wtake(256);
  c->ws_bytes = woff;
  c->oprm = p;
  c->ofn = fn;
  c->r_gt = GT; c->r_rpt = RPT;
  c->smem_bytes = smem;
  c->path = 6;
  c->planned = true;
  c->ws = nullptr;
  c->ws_given = 0;
  c->ran = false;
  return PCA_OK;
}

// fp64 storage (PCA_OPT_STORAGE = 1): the two-sweep streaming kernel instantiated on double (path 8)
int make_f64_plan(pca_ctx* c) {
  if (c->opt_path != 0 && c->opt_path != 1 && c->opt_path != 8) return PCA_EUNSUPPORTED;
  const long long M = c->M, N = c->N;
  const int sms = c->num_sms;
  const int g_min = (int)ceil_div(N, pca::kThreads);
  if (g_min > sms) return PCA_EUNSUPPORTED;
  int G = c->opt_ctas > 0 ? c->opt_ctas : sms;
  if (G < g_min) G = g_min;
  if (G > sms) G = sms;
  SolveParams g{};
  int tr = 0, rc = 0;
  const size_t smem = carve(c, 0, G, 1, &g, &tr, &rc, 8);
  if (smem > (size_t)c->smem_optin || tr != 32 || rc != 4) return PCA_EUNSUPPORTED;
  cudaError_t e = cudaFuncSetAttribute(pca::pca_solve_f64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin);   // per FUNCTION: the device maximum, so that contexts do not lower it for each other
  if (e != cudaSuccess) return cuda_fail(c, e);
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pca::pca_solve_f64_kernel, pca::kThreads, smem);
  if (e != cudaSuccess) return cuda_fail(c, e);
  if ((long long)per_sm * sms < g.G) return PCA_EUNSUPPORTED;
  pca::SolveParamsT<double> p{};
  p.M = M; p.N = N; p.K = c->K; p.eps = c->eps; p.max_iter = c->max_iter; p.algo = c->algo; p.test_mode = c->opt_test_mode;
  p.stag2 = c->opt_stag2; p.out_svd = c->opt_output; p.gs_passes = c->opt_gs_passes;
  p.G = g.G; p.Mb = g.Mb; p.Ns = g.Ns; p.Gs = g.Gs; p.slab_ld = 0; p.Npad = g.Npad; p.Kpad = g.Kpad;
  p.off_t = g.off_t; p.off_d = g.off_d; p.off_p = g.off_p; p.off_slice = g.off_slice; p.off_coef = g.off_coef;
  p.off_lam = g.off_lam; p.off_scr = g.off_scr; p.off_red = g.off_red; p.off_slab = g.off_slab;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = (size_t)round_up((long long)(off + bytes), 256); return o; };
  take((size_t)M * (size_t)N * 8);                                   // residual of eq. (4), column-major, double
  c->ws_off_ppart = take((size_t)p.G * p.Npad * 8);
  c->ws_off_apart = take((size_t)2 * p.Gs * p.Kpad * 8);
  c->ws_off_bpart = take((size_t)2 * p.G * p.Kpad * 8);
  c->ws_off_pvec = take((size_t)p.Npad * 8);
  c->ws_off_qpart = take((size_t)p.Gs * 8);
  c->ws_off_spart = take((size_t)p.G * 8);
  c->ws_off_bar = take(256);
  c->ws_bytes = off;
  c->prm64 = p;
  c->smem_bytes = smem;
  c->path = 8;
  c->planned = true;
  c->ws = nullptr;
  c->ws_given = 0;
  c->ran = false;
  return PCA_OK;
}

int make_plan(pca_ctx* c) {
  c->planned = false;
  if (c->opt_storage == 1) return make_f64_plan(c);
  // CGS2 (PCA_OPT_GS_PASSES = 2) is built into the two-sweep kernel only (paths 1, 2), whose pass has a separate phase
  // per projection; the single-sweep kernels fold the scores-side projection into the loads by linearity and have no
  // place for a second one.
  const bool cgs2 = c->opt_gs_passes > 1 && c->algo == PCA_ALGO_GS;
  if (cgs2 && c->opt_path >= 3) return PCA_EUNSUPPORTED;
  if (!cgs2 && ((c->opt_path == 0 && c->opt_trace == 0) || c->opt_path == 6)) {
    const int rc = make_one_plan(c);
    if (rc == PCA_OK || c->opt_path != 0) return rc;
    if (rc == PCA_ECUDA) return rc;
  }
  if (!cgs2 && (c->opt_path == 0 || c->opt_path == 5)) {
    const int rc = make_reg_plan(c);
    if (rc == PCA_OK || c->opt_path != 0) return rc;
    if (rc == PCA_ECUDA) return rc;
  }
  if (!cgs2 && (c->opt_path == 0 || c->opt_path == 3 || c->opt_path == 4 || c->opt_path == 7)) {
    const int rc = make_fused_plan(c, c->opt_path);
    if (rc == PCA_OK || c->opt_path != 0) return rc;
    if (rc == PCA_ECUDA) return rc;
  }
  const long long M = c->M, N = c->N;
  const int vec = (M % 4 == 0) ? 4 : 1;
  const int sms = c->num_sms;
  // every slice owner handles at most kThreads columns
  const int g_min = (int)ceil_div(N, pca::kThreads);
  if (g_min > sms) return PCA_EUNSUPPORTED;

  auto try_plan = [&](int resident, int G, SolveParams* p, const Variant** var, size_t* smem) -> bool {
    if (G < g_min) G = g_min;
    if (G > sms) G = sms;
    if (G < 1) G = 1;
    int tr, rc;
    *smem = carve(c, resident, G, vec, p, &tr, &rc);
    if (*smem > (size_t)c->smem_optin) return false;
    *var = find_variant(resident, vec, tr, rc);
    return *var != nullptr;
  };

  SolveParams p{};
  const Variant* var = nullptr;
  size_t smem = 0;
  bool ok = false;
  int path = 0;
  const int want_path = c->opt_path;
  if (want_path == 0 || want_path == 2) {
    // resident: a single CTA if the whole matrix fits comfortably, else one CTA per SM
    int G = c->opt_ctas > 0 ? c->opt_ctas : ((size_t)M * (size_t)N * 4 <= (size_t)160 * 1024 ? 1 : sms);
    ok = try_plan(1, G, &p, &var, &smem);
    if (!ok && c->opt_ctas == 0 && G != sms) ok = try_plan(1, sms, &p, &var, &smem);
    if (ok) path = 2;
    else if (want_path == 2) return PCA_EUNSUPPORTED;
  }
  if (!ok) {
    int G = c->opt_ctas > 0 ? c->opt_ctas : sms;
    ok = try_plan(0, G, &p, &var, &smem);
    if (!ok) return PCA_EUNSUPPORTED;
    path = 1;
  }
  // co-residency of the cooperative grid
  cudaError_t e = cudaFuncSetAttribute(var->fn, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin);   // per FUNCTION: the device maximum, so that contexts do not lower it for each other
  if (e != cudaSuccess) return cuda_fail(c, e);
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, var->fn, pca::kThreads, smem);
  if (e != cudaSuccess) return cuda_fail(c, e);
  if ((long long)per_sm * sms < p.G) return PCA_EUNSUPPORTED;

  p.M = M; p.N = N; p.K = c->K; p.eps = c->eps; p.max_iter = c->max_iter; p.algo = c->algo; p.test_mode = c->opt_test_mode; p.stag2 = c->opt_stag2; p.out_svd = c->opt_output;
  p.gs_passes = c->opt_gs_passes;
  // workspace layout: R first
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = (size_t)round_up((long long)(off + bytes), 256); return o; };
  take((size_t)M * (size_t)N * 4);
  c->ws_off_ppart = take((size_t)p.G * p.Npad * 4);
  c->ws_off_apart = take((size_t)2 * p.Gs * p.Kpad * 8);            // one buffer per Gram-Schmidt projection (CGS2: two)
  c->ws_off_bpart = take((size_t)2 * p.G * p.Kpad * 8);
  c->ws_off_pvec = take((size_t)p.Npad * 4);
  c->ws_off_qpart = take((size_t)p.Gs * 8);
  c->ws_off_spart = take((size_t)p.G * 8);
  c->ws_off_bar = take(256);
  c->ws_bytes = off;
  c->prm = p;
  c->variant = var;
  c->smem_bytes = smem;
  c->path = path;
  c->planned = true;
  c->ws = nullptr;  // a new plan invalidates a previously set workspace
  c->ws_given = 0;
  c->ran = false;
  return PCA_OK;
}

int pca_set_option_impl(pca_ctx* c, int option, int64_t value) {
  switch (option) {
    case PCA_OPT_PATH:
      if (value < 0 || value > 8) return PCA_EINVAL;
      c->opt_path = (int)value;
      break;
    case PCA_OPT_CTAS:
      if (value < 0 || value > c->num_sms) return PCA_EINVAL;
      c->opt_ctas = (int)value;
      break;
    case PCA_OPT_CENTER_MODE:
      if (value < 0 || value > 1) return PCA_EINVAL;
      c->opt_center_mode = (int)value;
      return PCA_OK;
    case PCA_OPT_OWNERS:
      if (value < 0 || value > c->num_sms) return PCA_EINVAL;
      c->opt_owners = (int)value;
      break;
    case PCA_OPT_KDIRECT:
      if (value < -1 || value > (1 << 30)) return PCA_EINVAL;
      c->opt_kdirect = (int)value;
      break;
    case PCA_OPT_TEST_MODE:
      if (value < 0 || value > 1) return PCA_EINVAL;
      c->opt_test_mode = (int)value;
      break;
    case PCA_OPT_TRACE:
      if (value < 0 || value > (1 << 24)) return PCA_EINVAL;
      c->opt_trace = (int)value;
      break;
    case PCA_OPT_STAGNATION:
      if (value < 0 || value > 1) return PCA_EINVAL;
      c->opt_stag2 = (int)value;
      break;
    case PCA_OPT_OUTPUT:
      if (value < 0 || value > 1) return PCA_EINVAL;
      c->opt_output = (int)value;
      break;
    case PCA_OPT_GS_PASSES:
      if (value < 1 || value > 2) return PCA_EINVAL;
      c->opt_gs_passes = (int)value;
      break;
    case PCA_OPT_RING_ROWS:
      if (value != 0 && value != 1 && value != 2 && value != 4) return PCA_EINVAL;
      c->opt_ring_rows = (int)value;
      break;
    case PCA_OPT_RING_SLOTS:
      if (value < 0 || value > 8) return PCA_EINVAL;
      c->opt_ring_slots = (int)value;
      break;
    case PCA_OPT_STORAGE:
      if (value < 0 || value > 1) return PCA_EINVAL;
      c->opt_storage = (int)value;
      break;
    case PCA_OPT_DEFER_S3:
      if (value < 0 || value > 1) return PCA_EINVAL;
      c->opt_defer_s3 = (int)value;
      break;
    default:
      return PCA_EINVAL;
  }
  return make_plan(c);
}


bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

extern "C" {

int pca_create(pca_ctx** out, int64_t M, int64_t N, int K, double eps, int max_iter, int algo) {
  if (!out) return PCA_EINVAL;
  *out = nullptr;
  if (M < 1 || N < 1 || K < 1 || (int64_t)K > N || !(eps >= 0.0) || max_iter < 1) return PCA_EINVAL;
  if (algo != PCA_ALGO_NIPALS && algo != PCA_ALGO_GS) return PCA_EINVAL;
  if (N > (int64_t)1 << 30 || M > (int64_t)1 << 40) return PCA_EUNSUPPORTED;
  pca_ctx* c = new (std::nothrow) pca_ctx();
  if (!c) return PCA_EINVAL;
  c->M = M; c->N = N; c->K = K; c->eps = eps; c->max_iter = max_iter; c->algo = algo;
  cudaError_t e = cudaGetDevice(&c->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device);
  int coop = 0;
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device);
  if (e != cudaSuccess || !coop) {
    delete c;
    return PCA_ECUDA;  // no CUDA device: there is no CPU fallback
  }
  const int rc = make_plan(c);
  if (rc != PCA_OK) {
    delete c;
    return rc;
  }
  *out = c;
  return PCA_OK;
}

int pca_set_option(pca_ctx* c, int option, int64_t value) {
  if (!c) return PCA_EINVAL;
  const pca_ctx saved = *c;                                      // a re-plan that fails leaves the context as it was
  const int rc = pca_set_option_impl(c, option, value);
  if (rc != PCA_OK) *c = saved;
  return rc;
}

int pca_get_info(const pca_ctx* c, int field, int64_t* value) {
  if (!c || !value || !c->planned) return PCA_EINVAL;
  if (c->path == 8) {                                              // fp64 two-sweep kernel
    switch (field) {
      case PCA_INFO_PATH: *value = 8; return PCA_OK;
      case PCA_INFO_CTAS: *value = c->prm64.G; return PCA_OK;
      case PCA_INFO_OWNERS: *value = c->prm64.Gs; return PCA_OK;
      case PCA_INFO_ROWS_PER_CTA: *value = c->prm64.Mb; return PCA_OK;
      case PCA_INFO_LAUNCHES_PER_RUN: *value = 1; return PCA_OK;
      case PCA_INFO_ROW_GROUP_THREADS: case PCA_INFO_RING_ROWS: case PCA_INFO_RING_SLOTS: case PCA_INFO_RUN_STATUS: *value = 0; return PCA_OK;
      default: break;
    }
  }
  switch (field) {
    case PCA_INFO_PATH: *value = c->path; break;
    case PCA_INFO_CTAS: *value = c->path == 6 ? 1 : c->path == 5 ? c->rprm.G : (c->path >= 3 ? c->fprm.G : c->prm.G); break;
    case PCA_INFO_OWNERS: *value = c->path == 6 ? 1 : c->path == 5 ? c->rprm.Gs : (c->path >= 3 ? c->fprm.Gs : c->prm.Gs); break;
    case PCA_INFO_THREADS: *value = c->path == 7 ? pca::kTmaThreads : pca::kThreads; break;
    case PCA_INFO_SMEM_BYTES: *value = (int64_t)c->smem_bytes; break;
    case PCA_INFO_ROWS_PER_CTA: *value = c->path == 6 ? c->oprm.M : c->path == 5 ? c->rprm.Mb : (c->path >= 3 ? c->fprm.Mb : c->prm.Mb); break;
    case PCA_INFO_LAUNCHES_PER_RUN: *value = c->path >= 3 ? 3 : 1; break;
    case PCA_INFO_ROW_GROUP_THREADS: *value = (c->path == 5 || c->path == 6) ? c->r_gt : (c->path >= 3 ? c->fprm.GT : 0); break;
    case PCA_INFO_RING_ROWS: *value = c->path == 7 ? c->ring_rows : 0; break;
    case PCA_INFO_RING_SLOTS: *value = c->path == 7 ? c->fprm.SG : 0; break;
    case PCA_INFO_NUM_SMS: *value = c->num_sms; break;
    case PCA_INFO_RUN_STATUS: {
      *value = 0;
      if (c->path >= 3 && c->path != 6 && c->ws && c->ran) {
        unsigned st = 0;
        if (cudaMemcpy(&st, static_cast<const unsigned char*>(c->ws) + c->ws_off_status, sizeof(st),
                       cudaMemcpyDeviceToHost) != cudaSuccess) return PCA_ECUDA;
        *value = (int64_t)st;
      }
      break;
    }
    default: return PCA_EINVAL;
  }
  return PCA_OK;
}

size_t pca_workspace_bytes(const pca_ctx* c) { return (c && c->planned) ? c->ws_bytes : 0; }

int pca_set_workspace(pca_ctx* c, void* dev, size_t bytes) {
  if (!c || !dev || !c->planned) return PCA_EINVAL;
  if ((reinterpret_cast<uintptr_t>(dev) & 255u) != 0) return PCA_EALIGN;
  if (bytes < c->ws_bytes) return PCA_EWORKSPACE;
  c->ws = dev;
  c->ws_given = bytes;
  c->ran = false;
  return PCA_OK;
}

int pca_center(pca_ctx* c, float* X, void* stream) {
  if (!c || !X) return PCA_EINVAL;
  if (!aligned16(X)) return PCA_EALIGN;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (c->opt_center_mode == 0) {
    const int grid = (int)(c->N < (long long)c->num_sms * 4 ? c->N : (long long)c->num_sms * 4);
    pca::pca_center_columns_kernel<<<grid, pca::kCenterThreads, 0, st>>>(X, c->M, (int)c->N, (c->M % 4 == 0) ? 1 : 0);
  } else {
    const long long grid = (c->M + 255) / 256;
    pca::pca_center_eq1_kernel<<<(unsigned)grid, 256, 0, st>>>(X, c->M, (int)c->N);
  }
  PCA_CUDA(c, cudaGetLastError());
  return PCA_OK;
}

int pca_center_f64(pca_ctx* c, double* X, void* stream) {
  if (!c || !X) return PCA_EINVAL;
  if (!aligned16(X)) return PCA_EALIGN;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (c->opt_center_mode == 0) {
    const int grid = (int)(c->N < (long long)c->num_sms * 4 ? c->N : (long long)c->num_sms * 4);
    pca::pca_center_columns_f64_kernel<<<grid, pca::kCenterThreads, 0, st>>>(X, c->M, (int)c->N);
  } else {
    const long long grid = (c->M + 255) / 256;
    pca::pca_center_eq1_f64_kernel<<<(unsigned)grid, 256, 0, st>>>(X, c->M, (int)c->N);
  }
  PCA_CUDA(c, cudaGetLastError());
  return PCA_OK;
}

int pca_run_f64(pca_ctx* c, const double* X, double* T, double* P, double* lambda, int32_t* iters, void* stream) {
  if (!c || !X || !T || !P || !lambda || !iters || !c->planned) return PCA_EINVAL;
  if (c->path != 8) return PCA_EINVAL;                             // needs PCA_OPT_STORAGE = 1
  if (!aligned16(X) || !aligned16(T) || !aligned16(P)) return PCA_EALIGN;
  if (!c->ws || c->ws_given < c->ws_bytes) return PCA_EWORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  unsigned char* ws = static_cast<unsigned char*>(c->ws);
  pca::SolveParamsT<double> p = c->prm64;
  p.X = X;
  p.R = reinterpret_cast<double*>(ws);
  p.Tm = T; p.P = P; p.lambda = lambda; p.iters = iters;
  p.Ppart = reinterpret_cast<double*>(ws + c->ws_off_ppart);
  p.Apart = reinterpret_cast<double*>(ws + c->ws_off_apart);
  p.Bpart = reinterpret_cast<double*>(ws + c->ws_off_bpart);
  p.pvec = reinterpret_cast<double*>(ws + c->ws_off_pvec);
  p.qpart = reinterpret_cast<double*>(ws + c->ws_off_qpart);
  p.spart = reinterpret_cast<double*>(ws + c->ws_off_spart);
  p.bar = reinterpret_cast<unsigned long long*>(ws + c->ws_off_bar);
  PCA_CUDA(c, cudaMemsetAsync(p.bar, 0, 256, st));
  void* args[] = {&p};
  PCA_CUDA(c, cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(pca::pca_solve_f64_kernel), dim3((unsigned)p.G),
                                          dim3(pca::kThreads), args, c->smem_bytes, st));
  c->ran = true;
  return PCA_OK;
}

int pca_residual_f64(const pca_ctx* c, const double** R) {
  if (!c || !R) return PCA_EINVAL;
  if (c->path != 8) return PCA_EINVAL;
  if (!c->ws || !c->ran) return PCA_EWORKSPACE;
  *R = reinterpret_cast<const double*>(c->ws);
  return PCA_OK;
}

int pca_run(pca_ctx* c, const float* X, float* T, float* P, float* lambda, int32_t* iters, void* stream) {
  if (!c || !X || !T || !P || !lambda || !iters || !c->planned) return PCA_EINVAL;
  if (c->path == 8) return PCA_EINVAL;                             // fp64 storage: pca_run_f64
  if (!aligned16(X) || !aligned16(T) || !aligned16(P)) return PCA_EALIGN;
  if (!c->ws || c->ws_given < c->ws_bytes) return PCA_EWORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  unsigned char* ws = static_cast<unsigned char*>(c->ws);
  if (c->path == 6) {
    OneParams p = c->oprm;
    p.Rrm = reinterpret_cast<float*>(ws + c->ws_off_rrm);
    p.T = T; p.P = P; p.lambda = lambda; p.iters = iters;
    const dim3 tgrid((unsigned)ceil_div(c->M, 32), (unsigned)ceil_div(p.ldr, 32));
    pca::pca_transpose_in_kernel<<<tgrid, 256, 0, st>>>(X, p.Rrm, c->M, p.N, p.ldr);   // R <- X
    PCA_CUDA(c, cudaGetLastError());
    c->ofn<<<1, pca::kThreads, c->smem_bytes, st>>>(p);
    PCA_CUDA(c, cudaGetLastError());
    const dim3 ogrid((unsigned)ceil_div(c->M, 32), (unsigned)ceil_div(c->N, 32));
    pca::pca_transpose_plain_kernel<<<ogrid, 256, 0, st>>>(p.Rrm, reinterpret_cast<float*>(ws), c->M, p.N, p.ldr);
    PCA_CUDA(c, cudaGetLastError());
    c->ran = true;
    return PCA_OK;
  }
  if (c->path == 5) {
    RegParams p = c->rprm;
    p.Rrm = reinterpret_cast<float*>(ws + c->ws_off_rrm);
    p.T = T; p.P = P; p.lambda = lambda; p.iters = iters;
    typedef unsigned long long u64;
    p.Qx = reinterpret_cast<u64*>(ws + c->ws_off_qx);
    p.SBx = reinterpret_cast<u64*>(ws + c->ws_off_sbx);
    p.Bx = reinterpret_cast<u64*>(ws + c->ws_off_bx);
    p.Ax = reinterpret_cast<u64*>(ws + c->ws_off_ax);
    p.Px = reinterpret_cast<u64*>(ws + c->ws_off_px);
    p.Nx = reinterpret_cast<u64*>(ws + c->ws_off_nx);
    p.Pfx = reinterpret_cast<u64*>(ws + c->ws_off_pfx);
    p.Nfx = reinterpret_cast<u64*>(ws + c->ws_off_nfx);
    p.status = reinterpret_cast<unsigned*>(ws + c->ws_off_status);
    p.trace = reinterpret_cast<unsigned long long*>(ws + c->ws_off_trace);
    PCA_CUDA(c, cudaMemsetAsync(ws + c->ws_off_xchg, 0, c->ws_xchg_bytes, st));   // sequence numbers start at 0
    if (p.trace_cap > 0) PCA_CUDA(c, cudaMemsetAsync(p.trace, 0, 8, st));
    const dim3 tgrid((unsigned)ceil_div(c->M, 32), (unsigned)ceil_div(p.ldr, 32));
    pca::pca_transpose_in_kernel<<<tgrid, 256, 0, st>>>(X, p.Rrm, c->M, p.N, p.ldr);   // R <- X
    PCA_CUDA(c, cudaGetLastError());
    void* rargs[] = {&p};
    PCA_CUDA(c, cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(c->rfn), dim3((unsigned)p.G), dim3(pca::kThreads),
                                            rargs, c->smem_bytes, st));
    const dim3 ogrid((unsigned)ceil_div(c->M, 32), (unsigned)ceil_div(c->N, 32));
    pca::pca_transpose_plain_kernel<<<ogrid, 256, 0, st>>>(p.Rrm, reinterpret_cast<float*>(ws), c->M, p.N, p.ldr);
    PCA_CUDA(c, cudaGetLastError());
    c->ran = true;
    return PCA_OK;
  }
  if (c->path >= 3) {
    FusedParams p = c->fprm;
    p.Rrm = reinterpret_cast<float*>(ws + c->ws_off_rrm);
    p.T = T; p.P = P; p.lambda = lambda; p.iters = iters;
    typedef unsigned long long u64;
    p.Qx = reinterpret_cast<u64*>(ws + c->ws_off_qx);
    p.SBx = reinterpret_cast<u64*>(ws + c->ws_off_sbx);
    p.Ax = reinterpret_cast<u64*>(ws + c->ws_off_ax);
    p.Px = reinterpret_cast<u64*>(ws + c->ws_off_px);
    p.Nx = reinterpret_cast<u64*>(ws + c->ws_off_nx);
    p.Pfx = reinterpret_cast<u64*>(ws + c->ws_off_pfx);
    p.Nfx = reinterpret_cast<u64*>(ws + c->ws_off_nfx);
    p.Pown = reinterpret_cast<float*>(ws + c->ws_off_pown);
    p.Wown = reinterpret_cast<float*>(ws + c->ws_off_wown);
    p.status = reinterpret_cast<unsigned*>(ws + c->ws_off_status);
    p.cnt = reinterpret_cast<unsigned*>(ws + c->ws_off_cnt);
    p.trace = reinterpret_cast<unsigned long long*>(ws + c->ws_off_trace);
    p.Vrm = reinterpret_cast<float*>(ws + c->ws_off_vrm);
    PCA_CUDA(c, cudaMemsetAsync(ws + c->ws_off_xchg, 0, c->ws_xchg_bytes, st));   // sequence numbers start at 0
    if (p.trace_cap > 0) PCA_CUDA(c, cudaMemsetAsync(p.trace, 0, 8, st));
    if (p.trace_cap > 0) PCA_CUDA(c, cudaMemsetAsync(p.trace + 1 + p.trace_cap, 0, (size_t)2 * p.G * 8, st));
    const dim3 tgrid((unsigned)ceil_div(c->M, 32), (unsigned)ceil_div(p.ldr, 32));
    pca::pca_transpose_in_kernel<<<tgrid, 256, 0, st>>>(X, p.Rrm, c->M, p.N, p.ldr);   // R <- X
    PCA_CUDA(c, cudaGetLastError());
    void* fargs[] = {&p};
    PCA_CUDA(c, cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(c->ffn), dim3((unsigned)p.G),
                                            dim3(c->path == 7 ? pca::kTmaThreads : pca::kThreads), fargs, c->smem_bytes, st));
    const dim3 ogrid((unsigned)ceil_div(c->M, 32), (unsigned)ceil_div(c->N, 32));
    pca::pca_transpose_out_kernel<<<ogrid, 256, 0, st>>>(p.Rrm, reinterpret_cast<float*>(ws),
                                                         T + (size_t)(c->K - 1) * (size_t)c->M,
                                                         P + (size_t)(c->K - 1) * (size_t)c->N,
                                                         c->opt_output ? lambda + (c->K - 1) : nullptr, c->M, p.N, p.ldr);
    PCA_CUDA(c, cudaGetLastError());
    c->ran = true;
    return PCA_OK;
  }
  SolveParams p = c->prm;
  p.X = X;
  p.R = reinterpret_cast<float*>(ws);
  p.Tm = T; p.P = P; p.lambda = lambda; p.iters = iters;
  p.Ppart = reinterpret_cast<float*>(ws + c->ws_off_ppart);
  p.Apart = reinterpret_cast<double*>(ws + c->ws_off_apart);
  p.Bpart = reinterpret_cast<double*>(ws + c->ws_off_bpart);
  p.pvec = reinterpret_cast<float*>(ws + c->ws_off_pvec);
  p.qpart = reinterpret_cast<double*>(ws + c->ws_off_qpart);
  p.spart = reinterpret_cast<double*>(ws + c->ws_off_spart);
  p.bar = reinterpret_cast<unsigned long long*>(ws + c->ws_off_bar);
  PCA_CUDA(c, cudaMemsetAsync(p.bar, 0, 256, st));
  void* args[] = {&p};
  PCA_CUDA(c, cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(c->variant->fn), dim3((unsigned)p.G),
                                          dim3(pca::kThreads), args, c->smem_bytes, st));
  c->ran = true;
  return PCA_OK;
}

int pca_residual(const pca_ctx* c, const float** R) {
  if (!c || !R) return PCA_EINVAL;
  if (c->path == 8) return PCA_EINVAL;
  if (!c->ws || !c->ran) return PCA_EWORKSPACE;
  *R = reinterpret_cast<const float*>(c->ws);
  return PCA_OK;
}

int pca_trace(const pca_ctx* c, const uint64_t** records, int64_t* capacity) {
  if (!c || !records || !capacity) return PCA_EINVAL;
  if (!c->planned || c->path < 3 || c->path == 6 || c->path == 8 || c->opt_trace <= 0) return PCA_EUNSUPPORTED;
  if (!c->ws || !c->ran) return PCA_EWORKSPACE;
  *records = reinterpret_cast<const uint64_t*>(static_cast<const unsigned char*>(c->ws) + c->ws_off_trace);
  *capacity = c->opt_trace;
  return PCA_OK;
}

int pca_fit_host(pca_ctx* c, const float* X_host, float* T_host, float* P_host, float* lambda_host,
                 int32_t* iters_host, void* stream) {
  if (!c || !X_host || !T_host || !P_host || !lambda_host || !iters_host || !c->planned) return PCA_EINVAL;
  if (c->path == 8) return PCA_EUNSUPPORTED;                       // host-buffer entry point: fp32 storage only
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const size_t xb = (size_t)c->M * (size_t)c->N * 4, tb = (size_t)c->M * c->K * 4, pb = (size_t)c->N * c->K * 4;
  // staging buffers (shape-dependent only; one pointer at a time so that a failed allocation is retried, not skipped)
  if (!c->hX) PCA_CUDA(c, cudaMalloc(reinterpret_cast<void**>(&c->hX), xb));
  if (!c->hT) PCA_CUDA(c, cudaMalloc(reinterpret_cast<void**>(&c->hT), tb));
  if (!c->hP) PCA_CUDA(c, cudaMalloc(reinterpret_cast<void**>(&c->hP), pb));
  if (!c->hLam) PCA_CUDA(c, cudaMalloc(reinterpret_cast<void**>(&c->hLam), (size_t)c->K * 4));
  if (!c->hIters) PCA_CUDA(c, cudaMalloc(reinterpret_cast<void**>(&c->hIters), (size_t)c->K * 4));
  if (!c->ws || c->ws == c->hWs) {
    // private workspace: a re-plan (pca_set_option) may have grown pca_workspace_bytes() since it was allocated
    if (c->hWs && c->hWs_bytes < c->ws_bytes) {
      PCA_CUDA(c, cudaStreamSynchronize(st));
      cudaFree(c->hWs);
      c->hWs = nullptr;
      c->hWs_bytes = 0;
      c->ws = nullptr;
    }
    if (!c->hWs) {
      PCA_CUDA(c, cudaMalloc(&c->hWs, c->ws_bytes));
      c->hWs_bytes = c->ws_bytes;
    }
    c->ws = c->hWs;
    c->ws_given = c->hWs_bytes;
  }
  PCA_CUDA(c, cudaMemcpyAsync(c->hX, X_host, xb, cudaMemcpyHostToDevice, st));
  int rc = pca_center(c, c->hX, stream);
  if (rc != PCA_OK) return rc;
  rc = pca_run(c, c->hX, c->hT, c->hP, c->hLam, c->hIters, stream);
  if (rc != PCA_OK) return rc;
  PCA_CUDA(c, cudaMemcpyAsync(T_host, c->hT, tb, cudaMemcpyDeviceToHost, st));
  PCA_CUDA(c, cudaMemcpyAsync(P_host, c->hP, pb, cudaMemcpyDeviceToHost, st));
  PCA_CUDA(c, cudaMemcpyAsync(lambda_host, c->hLam, (size_t)c->K * 4, cudaMemcpyDeviceToHost, st));
  PCA_CUDA(c, cudaMemcpyAsync(iters_host, c->hIters, (size_t)c->K * 4, cudaMemcpyDeviceToHost, st));
  unsigned run_status = 0;                                       // the exchange protocol's status word (paths 3-5)
  const bool has_status = c->path >= 3 && c->path != 6;
  if (has_status)
    PCA_CUDA(c, cudaMemcpyAsync(&run_status, static_cast<const unsigned char*>(c->ws) + c->ws_off_status, sizeof(run_status),
                                cudaMemcpyDeviceToHost, st));
  PCA_CUDA(c, cudaStreamSynchronize(st));
  if (has_status && run_status != 0) return PCA_EPROTOCOL;
  return PCA_OK;
}

void pca_destroy(pca_ctx* c) {
  if (!c) return;
  if (c->hX) cudaFree(c->hX);
  if (c->hT) cudaFree(c->hT);
  if (c->hP) cudaFree(c->hP);
  if (c->hLam) cudaFree(c->hLam);
  if (c->hIters) cudaFree(c->hIters);
  if (c->hWs) cudaFree(c->hWs);
  delete c;
}

const char* pca_strerror(int code) {
  switch (code) {
    case PCA_OK: return "ok";
    case PCA_EINVAL: return "invalid argument";
    case PCA_EALIGN: return "device pointer not sufficiently aligned";
    case PCA_ECUDA: return "CUDA runtime error (no device, or a launch/copy failed)";
    case PCA_EWORKSPACE: return "workspace missing or too small";
    case PCA_EUNSUPPORTED: return "shape not supported by this build";
    case PCA_EPROTOCOL: return "a cross-CTA exchange wait gave up: the results of this run are invalid";
    default: return "unknown error";
  }
}

int pca_last_cuda_error(const pca_ctx* c) { return c ? c->last_cuda : 0; }

}  // extern "C"
