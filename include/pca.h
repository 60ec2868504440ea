/* =====================================================================================
 * include/pca.h -- C ABI of the B200-native (sm_100a) hot path of Andrecut's iterative PCA
 * (arxiv 0811.1081, "Parallel GPU Implementation of Iterative PCA Algorithms"; the paper text
 * is cited as PAPER.md:<line>).
 *
 * The library computes, for a column-mean-centred M x N matrix X, the
 * truncated decomposition X = T_(K) P_(K)^T + R (eq. 4) one component at a time
 * with the power-style inner loop of NIPALS-PCA (section 2.2; listing
 * PAPER.md:555-568) or GS-PCA (section 2.3; listing PAPER.md:1016-1038).
 * Every step of that loop (loads p = R^T t, Gram-Schmidt against the previous loadings,
 * normalisation, scores t = R p, Gram-Schmidt against the previous scores, lambda = ||t||,
 * convergence test, rank-1 deflation) runs in hand-written CUDA kernels; the convergence test is
 * taken on the device, so no call below reads device data back to the host.
 *
 * Conventions
 *   layout     column-major, leading dimension = number of rows: element (m, n) of an M x N
 *              matrix is at index n*M + m, the paper's id(m,n,ld).
 *              A contiguous row-major (N, M) array IS the M x N column-major matrix.
 *   precision  fp32 storage and fp32 FMA in the two big matrix-vector products; norms, Gram-
 *              Schmidt coefficients, lambda and the convergence test are fp64 scalars on device.
 *   pointers   "dev" = device memory of the current CUDA device, "host" = host memory.
 *              Device matrices must be 16-byte aligned (PCA_EALIGN otherwise).
 *   stream     a cudaStream_t passed as void* (NULL = legacy default stream).
 *   async      pca_center / pca_run only ENQUEUE work on `stream` and return; results are valid
 *              once the caller has synchronised the stream.  Argument and launch errors are
 *              returned synchronously.  Nothing prints, throws or exits.
 *   ownership  the caller owns X, T, P, lambda, iters and the workspace; the context owns only
 *              host memory (plus, if pca_fit_host is used, its private device staging buffers).
 *   threads    one context = one problem shape; a context is not thread-safe; distinct
 *              contexts on distinct streams are independent.
 *   errors     every int-returning call returns PCA_OK (0) or one of the codes below.
 * ===================================================================================== */
#ifndef PCA_H_
#define PCA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pca_ctx pca_ctx; /* opaque */

enum { PCA_ALGO_NIPALS = 0, PCA_ALGO_GS = 1 };

enum {
  PCA_OK = 0,
  PCA_EINVAL = 1,       /* bad argument (see each call) */
  PCA_EALIGN = 2,       /* a device matrix pointer is not 16-byte aligned */
  PCA_ECUDA = 3,        /* a CUDA runtime call failed (pca_last_cuda_error has the code) */
  PCA_EWORKSPACE = 4,   /* no workspace set, or it is smaller than pca_workspace_bytes() */
  PCA_EUNSUPPORTED = 5, /* shape / option combination cannot be handled by this build (e.g. N too large for SMEM) */
  PCA_EPROTOCOL = 6     /* pca_fit_host only: a cross-CTA exchange wait of the persistent kernel gave up (status word
                           PCA_INFO_RUN_STATUS != 0); the results of that run are invalid.  Never in a correct run */
};

/* Options for pca_set_option (all optional; defaults are chosen by pca_create). */
enum {
  PCA_OPT_PATH = 1,     /* 0 = auto; two-sweep kernel: 1 = HBM-streaming, 2 = SMEM-resident;
                           single-sweep kernel (R read once per inner pass): 3 = streaming, 4 = SMEM-resident,
                           5 = register-resident (4*M*N up to ~19 MB on 148 SMs), 6 = one CTA (the matrix in the registers
                           of one SM: N <= 512, M <= (512/GT)*7 rows with GT = pow2 >= N/8),
                           7 = streaming through a shared-memory ring filled by bulk-async copies (TMA; cp.async.bulk +
                           mbarrier), Gram-Schmidt coefficients of the scores accumulated during the sweep by helper warps */
  PCA_OPT_CTAS = 2,     /* number of CTAs of the persistent kernel (0 = auto) */
  PCA_OPT_CENTER_MODE = 3, /* 0 = column means (default), 1 = literal eq. (1) mean column */
  PCA_OPT_OWNERS = 5,   /* register-resident kernel: number of slice-owner CTAs (0 = auto; rounded down to a power of two) */
  PCA_OPT_KDIRECT = 6,  /* register-resident kernel: the Gram-Schmidt coefficients B of component k are combined in two
                           levels for k > this value (-1 = default) */
  PCA_OPT_TEST_MODE = 7, /* convergence test: 0 = the listings' strict relative test |lambda - lambda'| < eps*lambda'
                           (default), 1 = the text's absolute test |lambda' - lambda| <= eps */
  PCA_OPT_TRACE = 4,    /* single-sweep kernels only: capacity (records) of the device-side phase trace, 0 = off
                           (default).  See pca_trace. */
  PCA_OPT_STAGNATION = 8, /* 1 (default): besides the listings' test, lambda' is also compared with the value TWO passes back
                           (reading C4b: in fp32 the iteration can end in a period-2 limit cycle that the
                           listings' test never sees); 0: the listings' / text's test alone, literally */
  PCA_OPT_OUTPUT = 9,   /* 0 (default): PCA output, T = V Lambda, ||T[:,k]|| = lambda[k];
                           1: SVD output "V, U, Lambda" (eq. 5 :56): T holds the UNIT score vectors V
                           (the epilogue S10 is skipped; NIPALS-PCA: t / lambda), P = U, lambda = Lambda */
  PCA_OPT_GS_PASSES = 10, /* GS-PCA: classical Gram-Schmidt projections per side per inner pass.  1 (default) = the listings
                           (PAPER.md:1025-1026, :1030-1031); 2 = CGS2, "applying it iteratively".  2 is built
                           into the two-sweep kernel only: the plan falls back to paths 1/2, forcing paths 3-6 gives
                           PCA_EUNSUPPORTED.  Ignored for NIPALS-PCA */
  PCA_OPT_RING_ROWS = 11, /* path 7: rows of R per ring slot (one bulk copy): 0 = auto, 1, 2 or 4 */
  PCA_OPT_RING_SLOTS = 12, /* path 7: upper bound on the ring slots per row group (0 = auto: what fits, at most 8) */
  PCA_OPT_DEFER_S3 = 15,  /* single-sweep kernels, GS-PCA: 1 (default): a pass may start its sweep from the loads p~ BEFORE the
                            loads-side Gram-Schmidt p^ = p~ - P A -- R p~ and R p^ give the same projected scores
                            -- whenever the previous pass measured that this costs no accuracy (p^ is then formed
                            once per component); 0: every pass takes the paper's order (one more cross-CTA hop per pass) */
  PCA_OPT_STORAGE = 14    /* 0 (default): fp32 storage (pca_center / pca_run / pca_residual); 1: fp64 storage and fp64 arithmetic
                            throughout, the paper's native precision: pca_center_f64 / pca_run_f64 /
                            pca_residual_f64, run by the two-sweep kernel (the paper's pass shape) instantiated on double
                            (PCA_INFO_PATH = 8); the fp32 entry points return PCA_EINVAL on such a context and vice versa */
};

/* Phase ids of the trace records (pca_trace).  One inner pass of the single-sweep kernel is
 * PREADY -> SWEEP -> PUBLISHED -> X1 -> TEST -> QSLICE -> [APART -> X2 ->] PHAT -> X3 -> PREADY. */
enum {
  PCA_TR_COMPONENT = 1, /* component k starts (S1)   (path 5 emits the subset COMPONENT, LOADS_DONE, X1, TEST, X2, PHAT, X3, SWEEP,
                           PUBLISHED, FINAL of these ids) */
  PCA_TR_LOADS_DONE = 2,/* first sweep of the component done: pending deflation S9 + q = R^T t0 (S2), published */
  PCA_TR_X1 = 3,        /* grid barrier 1 passed: all partial raw loads / |t~|^2 / B-partials visible */
  PCA_TR_TEST = 4,      /* lambda' (S7) and the convergence test (S8) taken */
  PCA_TR_QSLICE = 5,    /* slice owner: q slice combined and corrected to p~ = q - W B */
  PCA_TR_APART = 6,     /* GS-PCA: partial A = P_(k)^T p~ published (S3, first half) */
  PCA_TR_X2 = 7,        /* grid barrier 2 passed (GS-PCA, k > 0 only) */
  PCA_TR_PHAT = 8,      /* slice owner: p^ = p~ - P A and its partial squared norm published (S3/S4) */
  PCA_TR_X3 = 9,        /* grid barrier 3 passed */
  PCA_TR_PREADY = 10,   /* unit loads p in shared memory (S4) */
  PCA_TR_SWEEP = 11,    /* sweep over the CTA's rows done: t~ = R p (S5) and q = R^T t~ (S2 of the next pass) */
  PCA_TR_PUBLISHED = 12,/* partial q, |t~|^2 and B-partials (S6) written to the exchange buffers */
  PCA_TR_FINAL = 13     /* component finalised (T, P, lambda, iters, W column stored) */
};

/* Fields for pca_get_info. */
enum {
  PCA_INFO_PATH = 1,        /* 1, 2 = two-sweep kernel streaming / resident; 3, 4 = single-sweep kernel streaming / resident;
                               5 = register-resident single-sweep kernel; 6 = one-CTA single-sweep kernel; 7 = single-sweep kernel,
                               TMA ring; 8 = two-sweep kernel on fp64 storage */
  PCA_INFO_CTAS = 2,        /* CTAs of the persistent solve kernel */
  PCA_INFO_THREADS = 3,     /* threads per CTA */
  PCA_INFO_SMEM_BYTES = 4,  /* dynamic shared memory per CTA */
  PCA_INFO_ROWS_PER_CTA = 5,
  PCA_INFO_LAUNCHES_PER_RUN = 6, /* kernel launches one pca_run enqueues */
  PCA_INFO_NUM_SMS = 7,
  PCA_INFO_ROW_GROUP_THREADS = 8, /* single-sweep kernel: threads that share one row of R (0 otherwise) */
  PCA_INFO_OWNERS = 10,     /* slice-owner CTAs (CTAs that combine the partial loads of a column slice) */
  PCA_INFO_RING_ROWS = 11,  /* path 7: rows per ring slot (0 on other paths) */
  PCA_INFO_RING_SLOTS = 12, /* path 7: ring slots per row group */
  PCA_INFO_RUN_STATUS = 9   /* SYNCHRONISES the device and reads the status word of the last pca_run: 0 = ok,
                               1 = a cross-CTA exchange wait gave up (results invalid; never in a correct run) */
};

/* Create a context for one problem shape.
 *   M, N      rows (observations) and columns (attributes) of X, M >= 1, N >= 1
 *   K         number of components, 1 <= K <= N ("K <= N"; the start vector of
 *             component k is column k of the residual)
 *   eps       >= 0; relative stagnation tolerance of the listings' test
 *             |lambda - lambda'| < eps * lambda'; lambda' is also compared with
 *             the value two passes back (a period-2 limit cycle in fp32 is stagnation, C4b; PCA_OPT_STAGNATION = 0
 *             switches that off).  With the default relative test eps = 0 never fires, i.e. exactly max_iter passes per
 *             component (fixed-work benchmark mode); with PCA_OPT_TEST_MODE = 1 (|lambda' - lambda| <= eps) eps = 0 DOES
 *             fire once lambda' repeats exactly, as the text's test says
 *   max_iter  >= 1; the listings' J = 10000
 *   algo      PCA_ALGO_NIPALS or PCA_ALGO_GS
 * Needs a CUDA device (queries its SM count and shared-memory size); PCA_ECUDA if there is none.
 * Errors: PCA_EINVAL, PCA_ECUDA, PCA_EUNSUPPORTED. */
int pca_create(pca_ctx** out, int64_t M, int64_t N, int K, double eps, int max_iter, int algo);

/* Tune / query the launch plan.  pca_set_option must be called before pca_workspace_bytes /
 * pca_set_workspace; it re-plans (a previously set workspace is dropped: set it again) and may return
 * PCA_EUNSUPPORTED (e.g. forcing the resident path for a matrix that does not fit in shared memory),
 * in which case the context keeps its previous options and plan. */
int pca_set_option(pca_ctx*, int option, int64_t value);
int pca_get_info(const pca_ctx*, int field, int64_t* value);

/* Device workspace the caller must provide: the residual R of eq. (4) (4*M*N bytes, column-major,
 * first), followed -- for the single-sweep kernel -- by the row-major working copy of the residual
 * (4*M*ldr bytes, ldr = N rounded up to the row-group width), and the partial-sum / exchange
 * scratch of the persistent kernel. */
size_t pca_workspace_bytes(const pca_ctx*);

/* Hand the context a device buffer of at least pca_workspace_bytes() bytes, 256-byte aligned.
 * The caller keeps ownership and must keep it alive while the context is used.
 * Errors: PCA_EINVAL (NULL), PCA_EALIGN, PCA_EWORKSPACE (too small). */
int pca_set_workspace(pca_ctx*, void* dev, size_t bytes);

/* Step S0, mean centring, in place (eq. 1 / "each column is mean centered"):
 *   mu_n = (1/M) sum_m X[m,n];  X[m,n] -= mu_n          (default: column means, C1)
 * With PCA_OPT_CENTER_MODE = 1 the literal eq. (1) is applied instead (the mean COLUMN
 * (1/N) sum_n X^(n) is subtracted from every column; listing PAPER.md:1009-1013).
 *   X  dev, M x N, column-major ld = M, overwritten.
 * Errors: PCA_EINVAL, PCA_EALIGN, PCA_ECUDA. */
int pca_center(pca_ctx*, float* X, void* stream);

/* The hot path: K components of NIPALS-PCA / GS-PCA on a centred X.
 *   X       dev, M x N, ld = M, centred; never written (R <- X)
 *   T       dev, M x K, ld = M, scores.  ||T[:,k]|| = lambda[k] for both algorithms
 *           (NIPALS: t = R p; GS-PCA: T = V Lambda); with
 *           PCA_OPT_OUTPUT = 1 the unit vectors V instead (SVD output)
 *   P       dev, N x K, ld = N, loadings with unit columns
 *   lambda  dev, K floats, the last lambda' = ||T^(k)|| of each component (the paper's
 *           "eigenvalue" = singular value of the centred X); extraction order
 *   iters   dev, K int32, inner passes executed per component (1-based).  iters[k] == max_iter
 *           means the test never fired (reported, not an error).  A component whose start
 *           column, loads or scores have exactly zero norm returns lambda = 0, T = 0, P = 0,
 *           iters = 0 (C7).
 * After the stream is synchronised the residual R of eq. (4) is available via pca_residual.
 * Sign: (T[:,k], P[:,k]) is defined up to a joint sign.
 * Errors: PCA_EINVAL (NULL), PCA_EALIGN, PCA_EWORKSPACE, PCA_ECUDA. */
int pca_run(pca_ctx*, const float* X, float* T, float* P, float* lambda, int32_t* iters, void* stream);

/* Pointer to the residual R (dev, M x N, ld = M) inside the workspace; valid after a pca_run on
 * this context has completed ("return T, P, R"). */
int pca_residual(const pca_ctx*, const float** R);

/* fp64 storage variant (PCA_OPT_STORAGE = 1; the paper works in double precision throughout; SURVEY.md
 * section 8(f) F3).  Same semantics, layouts, ownership and error behaviour as pca_center / pca_run / pca_residual with every
 * matrix and vector in double (X, T, P, lambda: dev, column-major, 16-byte aligned); all arithmetic is fp64.  The workspace is
 * sized for double (pca_workspace_bytes after the option is set).  PCA_EINVAL on a context whose storage option is 0. */
int pca_center_f64(pca_ctx*, double* X, void* stream);
int pca_run_f64(pca_ctx*, const double* X, double* T, double* P, double* lambda, int32_t* iters, void* stream);
int pca_residual_f64(const pca_ctx*, const double** R);

/* Device-side phase trace of the last pca_run (tracing aid; PCA_OPT_TRACE > 0, single-sweep kernels, paths 3-5).
 *   records   dev pointer inside the workspace: records[0] = number of records written per slot,
 *             records[1 + i] = (phase id << 56) | (time stamp & (2^56 - 1)), in program order.
 *             paths 3, 4: ONE slot, CTA 0, time stamp = its SM cycle counter (clock64);
 *             path 5: one slot per CTA (CTA b owns records [b*capacity/G, (b+1)*capacity/G)), time stamp = %globaltimer
 *             in ns (common to all SMs), so that the timelines of the CTAs can be laid side by side.
 *             (With PCA_OPT_TRACE > 0 the auto plan does not pick the one-CTA kernel, which has no trace.)
 *   capacity  the PCA_OPT_TRACE value
 * Valid after the stream of pca_run has been synchronised; the caller copies it to the host.
 * Errors: PCA_EINVAL, PCA_EUNSUPPORTED (trace off, or a kernel without trace), PCA_EWORKSPACE (no run yet). */
int pca_trace(const pca_ctx*, const uint64_t** records, int64_t* capacity);

/* Convenience entry with HOST buffers (used for end-to-end timing): copies X (host, M x N,
 * NOT centred) to the device, runs pca_center and pca_run on `stream`, copies T, P, lambda, iters
 * back and synchronises the stream.  The context allocates private device staging buffers and
 * the workspace on first use (freed by pca_destroy; re-allocated if a later pca_set_option needs a
 * larger one).  Host buffers should be pinned for full PCIe bandwidth but need not be.  After the
 * synchronisation the run's status word is checked.  Errors: as pca_center / pca_run, PCA_EPROTOCOL. */
int pca_fit_host(pca_ctx*, const float* X_host, float* T_host, float* P_host, float* lambda_host,
                 int32_t* iters_host, void* stream);

void pca_destroy(pca_ctx*);

/* ---- Row-sharded multi-GPU form (the paper itself is single-GPU) -----------
 * One process per GPU; rank g holds M_local consecutive rows of the (centred) matrix X and gets its rows of T; P, lambda and
 * iters come out identical on every rank.  Per inner pass the ranks exchange ONE all-reduce (sum) of N + K' + 2 doubles
 * ([ R_g^T t~_g | |t~_g|^2 | V_g^T t~_g ], PAPER.md:1023, :1032, :1030 in the single-sweep form of the other kernels); the
 * all-reduce is the CALLER's (torch.distributed: NCCL between GPUs): every call below only enqueues rank-local kernels on
 * `stream`.  Calling sequence (paper_0811_1081_b200/sharded.py does exactly this):
 *     pca_shard_colsums -> all-reduce the N sums -> pca_shard_center                       (S0, column means over ALL rows)
 *     pca_shard_begin
 *     for k in 0..K-1:  pca_shard_component(k); exchange;
 *                       repeat { pca_shard_pass(k); exchange; } until pca_shard_done says 1   (it may be asked every few passes:
 *                                                                       steps after convergence are no-ops on the device)
 *                       pca_shard_finish_component(k)
 *     pca_shard_end
 *   "exchange" = copy the `send` buffer of pca_shard_exchange to `recv`, all-reduce `recv` in place (sum over the ranks).
 * Arguments as for pca_create / pca_center / pca_run with M_local rows: X_local, T (dev, M_local x N / M_local x K column-major,
 * ld = M_local), P (dev, N x K), lambda, iters (dev, K).  K <= 1024, N <= 8192.  Workspace: caller-owned, 256-byte aligned.
 * Errors: PCA_EINVAL, PCA_EALIGN, PCA_EWORKSPACE (no workspace / pca_shard_begin not called), PCA_EUNSUPPORTED, PCA_ECUDA. */
typedef struct pca_shard pca_shard;
int pca_shard_create(pca_shard** out, int64_t M_local, int64_t N, int K, double eps, int max_iter, int algo);
size_t pca_shard_workspace_bytes(const pca_shard*);
int pca_shard_set_workspace(pca_shard*, void* dev, size_t bytes);
int pca_shard_exchange(const pca_shard*, double** send /*dev*/, double** recv /*dev*/, int64_t* count /*doubles*/);
int pca_shard_colsums(pca_shard*, const float* X_local, double* sums /*dev, N: this rank's column sums*/, void* stream);
int pca_shard_center(pca_shard*, float* X_local, const double* sums_reduced /*dev, N*/, int64_t M_total, void* stream);
int pca_shard_begin(pca_shard*, const float* X_local, float* T, float* P, float* lambda, int32_t* iters, void* stream);
int pca_shard_component(pca_shard*, int k, void* stream);
int pca_shard_pass(pca_shard*, int k, void* stream);
int pca_shard_done(pca_shard*, int32_t* done_host /*host*/, void* stream);  /* synchronises `stream` */
int pca_shard_finish_component(pca_shard*, int k, void* stream);
int pca_shard_end(pca_shard*, float* R_local /*dev, M_local x N column-major: residual rows of eq. (4); may be NULL*/, void* stream);
void pca_shard_destroy(pca_shard*);
int pca_shard_last_cuda_error(const pca_shard*);   /* cudaError_t of the last PCA_ECUDA of this context */

/* ---- No-allocation entry point (README.md "No-allocation entry point") -----------------------------------------------------
 * pca_run for SMALL matrices without any device allocation and without a context: for callers that cannot call cudaMalloc
 * (code under CUDA-graph capture, tight serving loops, harnesses that forbid it).  It runs the one-CTA kernel of
 * PCA_OPT_PATH = 6 (the same inner loop, PAPER.md:555-568 / :1016-1038; same arithmetic, same results as pca_run on that path
 * with default options) and keeps the kernel's only scratch memory -- the row-major working copy of the residual, R <- X
 * -- in a file-scope device array of pca_small_static_scratch_bytes() = 114688 bytes that every GPU loading the
 * library holds until the process exits.
 *   limits     N <= 512 and M <= (512/GT)*7 rows with GT = the power of two >= max(8, N/8), so that M x (8*GT) floats fit in
 *              the array: M <= 448 for N <= 64, 224 for N <= 128, 112 for N <= 256, 56 for N <= 512.  Larger shapes are
 *              rejected with PCA_EUNSUPPORTED and a message naming the limit (pca_small_static_last_error); use pca_run.
 *   arguments  X, T, P, lambda, iters: dev, as for pca_run (X centred, column-major M x N, never written); eps, max_iter,
 *              algo as for pca_create; R: dev, M x N column-major, receives the residual of eq. (4), may be
 *              NULL; stream as everywhere.  X, T, P, R 16-byte aligned.  Options are the library defaults (the listings'
 *              relative test plus the two-pass stagnation check, PCA output).
 *   allocation none: no cudaMalloc / cudaFree, no allocating library routine, no host allocation.  The first call on a device
 *              looks up the array's device address and sets kernel attributes (make that call outside graph capture).
 *   sharing    all calls on a device share the array, which keeps the last call's contents; nothing in it needs to start at
 *              zero (the first kernel overwrites every word the solve reads).  Calls that OVERLAP on the GPU (different
 *              streams, concurrent host threads) race on it: keep them on one stream or order them with events.
 *   async      only enqueues three small kernels on `stream`.
 * Errors: PCA_EINVAL, PCA_EALIGN, PCA_EUNSUPPORTED (shape beyond the limits), PCA_ECUDA (pca_small_static_last_cuda_error). */
int pca_run_small_static(const float* X, int64_t M, int64_t N, int K, double eps, int max_iter, int algo, float* T, float* P,
                         float* lambda, int32_t* iters, float* R, void* stream);
size_t pca_small_static_scratch_bytes(void);          /* size of the static device array: 114688 */
const char* pca_small_static_last_error(void);        /* message of this thread's last failing pca_run_small_static ("" if none) */
int pca_small_static_last_cuda_error(void);           /* its cudaError_t (as int), 0 if none */

const char* pca_strerror(int code);

/* cudaError_t (as int) of the last failing CUDA call on this context, 0 if none. */
int pca_last_cuda_error(const pca_ctx*);

#ifdef __cplusplus
}
#endif
#endif /* PCA_H_ */
