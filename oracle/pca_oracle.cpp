// =====================================================================================
// oracle/pca_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, double-precision CPU restatement of the two iterative PCA algorithms of
//   M. Andrecut, "Parallel GPU Implementation of Iterative PCA Algorithms"
//   (arxiv 0811.1081; text in /root/reference/PAPER.md, cited below as PAPER.md:<line>).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may load this library.  It shares no code, header, table or helper with the CUDA path
// (paper_0811_1081_b200/csrc) and includes no CUDA header.
//
// What it follows, statement by statement:
//   * NIPALS-PCA : PAPER.md:36-47 (section 2.2 pseudo-code) in the statement order of the
//                  paper's own listing, Appendix 2.
//   * GS-PCA     : PAPER.md:60-90 (section 2.3 pseudo-code, partly garbled) in the statement
//                  order of Appendix 4.
//   * centring   : "each column is mean centered" -- DESIGN.md reading C1;
//                  the literal eq. (1) (listing PAPER.md:1009-1013: subtract the
//                  mean COLUMN) is offered as oracle_center_eq1.
//   * BLAS steps : gemv eq. (6), nrm2 eq. (8), ger eq. (9)
//                  written out as plain loops, no blocking, no reordering.
//   * Jacobi     : textbook cyclic Jacobi eigenvalue iteration (Golub & Van Loan, the paper's
//                  own reference [Golub et al., 1996]); used only by the tests as the
//                  brute-force pin "eigen-decomposition of X^T X on tiny inputs".
//
// Readings of silent / ambiguous points (DESIGN.md section 3 lists them all):
//   C3  convergence test is the listings' strict relative one: |lambda - lambda'| < eps*lambda'
//       (PAPER.md:566, :1034), not the text's absolute one.
//   C5  at most max_iter passes (listing `for(j=0;j<J;j++)`).
//   C6  start vector = column k of the DEFLATED residual.
//   C7  a component whose start column, loads or scores have exactly zero norm is returned
//       as lambda=0, T=0, P=0, iters=0 (the paper divides by zero there).
//
// Parity pins (tests/test_oracle_pins.py): prescribed spectrum (noise-free), Jacobi on X^T X,
// numpy SVD, energy identity, decomposition identity eq. (4), orthogonality, hand-derived
// worked examples under tests/golden/ (NIPALS 3x2, GS-PCA 3x3 with one pass per component), control-
// flow special cases.  tests/test_oracle_mutants.py types one plausible mistake at a time into a
// copy of this file (wrong sign / dropped step / k-1 columns in either Gram-Schmidt step, undeflated
// start vector, eps scaled by the old lambda, ...) and checks that a pin fails for each.  No function
// here is "parity unpinned".
//
// Layout everywhere: column-major, leading dimension = number of rows, the paper's
// id(m,n,ld) = n*ld + m.
//
// OpenMP is used only as `parallel for schedule(static)` over independent outputs; every
// output element is summed by one thread in a fixed order, so results do not depend on the
// number of threads.
// =====================================================================================
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

inline int64_t id(int64_t m, int64_t n, int64_t ld) { return n * ld + m; }

// nrm2, eq. (8) PAPER.md:132 (sum over m = 0..len-1; the paper's upper limit M is a typo).
double nrm2(const double* x, int64_t len) {
  double s = 0.0;
  for (int64_t i = 0; i < len; ++i) s += x[i] * x[i];
  return std::sqrt(s);
}

// y = A^T x, eq. (6) PAPER.md:115 with alpha=1, beta=0.  A is rows x cols, ld = rows.
void gemv_t(const double* A, int64_t rows, int64_t cols, const double* x, double* y) {
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < cols; ++n) {
    double s = 0.0;
    for (int64_t m = 0; m < rows; ++m) s += A[id(m, n, rows)] * x[m];
    y[n] = s;
  }
}

// y = A x, eq. (6) PAPER.md:115 with alpha=1, beta=0.  Every y[m] is summed over n = 0..cols-1
// in that order; rows are split into static blocks only to use the cores.
void gemv_n(const double* A, int64_t rows, int64_t cols, const double* x, double* y) {
  const int64_t blk = 512;
  const int64_t nblk = (rows + blk - 1) / blk;
#pragma omp parallel for schedule(static)
  for (int64_t b = 0; b < nblk; ++b) {
    const int64_t m0 = b * blk, m1 = (m0 + blk < rows) ? m0 + blk : rows;
    for (int64_t m = m0; m < m1; ++m) y[m] = 0.0;
    for (int64_t n = 0; n < cols; ++n) {
      const double xn = x[n];
      const double* a = A + id(0, n, rows);
      for (int64_t m = m0; m < m1; ++m) y[m] += a[m] * xn;
    }
  }
}

// A <- alpha x y^T + A, eq. (9) PAPER.md:139.
void ger(double* A, int64_t rows, int64_t cols, double alpha, const double* x, const double* y) {
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < cols; ++n) {
    const double ay = alpha * y[n];
    double* a = A + id(0, n, rows);
    for (int64_t m = 0; m < rows; ++m) a[m] += ay * x[m];
  }
}

}  // namespace

extern "C" {

// Threads the OpenMP loops will use (bench.py reports it as cpu_baseline.cores).
int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

// Column-mean centring (reading C1): mu_n = (1/M) sum_m X[m,n];  X[m,n] -= mu_n.
// "each column is mean centered" with columns = attributes.
int oracle_center(double* X, int64_t M, int64_t N) {
  if (!X || M < 1 || N < 1) return 1;
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < N; ++n) {
    double s = 0.0;
    for (int64_t m = 0; m < M; ++m) s += X[id(m, n, M)];
    const double mu = s / (double)M;
    for (int64_t m = 0; m < M; ++m) X[id(m, n, M)] -= mu;
  }
  return 0;
}

// Literal eq. (1), PAPER.md:23 and listing PAPER.md:1009-1013: U = sum_n X^(n) (a length-M
// column), then every column gets -U/N.  Documented non-default mode (C1).
int oracle_center_eq1(double* X, int64_t M, int64_t N) {
  if (!X || M < 1 || N < 1) return 1;
  std::vector<double> U(X, X + M);                                  // Dcopy
  for (int64_t n = 1; n < N; ++n)                                   // Daxpy(+1)
    for (int64_t m = 0; m < M; ++m) U[m] += X[id(m, n, M)];
  for (int64_t n = 0; n < N; ++n)                                   // Daxpy(-1/N)
    for (int64_t m = 0; m < M; ++m) X[id(m, n, M)] += (-1.0 / (double)N) * U[m];
  return 0;
}

// NIPALS-PCA (algo = 0) and GS-PCA (algo = 1).
//   X      in : M x N, centred, col-major ld = M (never written)
//   T      out: M x K scores, ld = M.  ||T[:,k]|| = lambda[k] for both algorithms
//               (NIPALS: t = R p un-normalised; GS-PCA: T = V Lambda)
//   P      out: N x K loadings, ld = N, unit columns
//   lambda out: K, last lambda' of each component (= singular value estimate)
//   iters  out: K, inner passes executed (1-based); == max_iter means the test never fired
//   R      out: M x N residual after K deflations ("return T, P, R"); may be NULL
// returns 0, or 1 on invalid arguments.
//   test_mode  0: the listings' strict relative test |lambda - lambda'| < eps*lambda' (reading C3, default)
//              1: the text's / pseudo-code's absolute test |lambda' - lambda| <= eps
//   gs_passes  GS-PCA: classical Gram-Schmidt projections per side per inner pass.  1 = the listings (PAPER.md:1025-1026,
//              :1030-1031; reading C9, default); 2 = "applying it iteratively" (CGS2): each projection is simply
//              done twice in a row.  In exact arithmetic the second projection is the identity.
int oracle_pca_ex2(const double* X, int64_t M, int64_t N, int K, double eps, int max_iter, int algo, int test_mode,
                   int gs_passes, double* T, double* P, double* lambda, int32_t* iters, double* R_out) {
  if (!X || !T || !P || !lambda || !iters) return 1;
  if (M < 1 || N < 1 || K < 1 || K > N || !(eps >= 0.0) || max_iter < 1) return 1;
  if (algo != 0 && algo != 1) return 1;
  if (test_mode != 0 && test_mode != 1) return 1;
  if (gs_passes != 1 && gs_passes != 2) return 1;
  const bool gs = (algo == 1);

  std::vector<double> Rv((size_t)M * (size_t)N);
  double* R = Rv.data();
  std::memcpy(R, X, sizeof(double) * (size_t)M * (size_t)N);         // R <- X
  std::vector<double> coef((size_t)(K > 1 ? K : 1));                 // A / B

  for (int k = 0; k < K; ++k) {
    double* t = T + id(0, k, M);   // GS-PCA: holds the unit vector V^(k) until the final scaling
    double* p = P + id(0, k, N);
    for (int64_t m = 0; m < M; ++m) t[m] = R[id(m, k, M)];           // T^(k) <- R^(k)
    double lam = 0.0;                                                // lambda = 0
    double lam_new = 0.0;
    int it = 0;
    bool degenerate = (nrm2(t, M) == 0.0);                           // reading C7
    for (int j = 0; j < max_iter && !degenerate; ++j) {              // PAPER.md:561,:1022 (C5)
      gemv_t(R, M, N, t, p);                                         // P^(k) <- R^T T^(k)
      for (int rep = 0; gs && k > 0 && rep < gs_passes; ++rep) {
        gemv_t(P, N, k, p, coef.data());                             // A <- U_(k)^T U^(k)
        for (int i = 0; i < k; ++i) {                                // U^(k) <- U^(k) - U_(k) A
          const double a = coef[i];
          const double* pi = P + id(0, i, N);
          for (int64_t n = 0; n < N; ++n) p[n] -= pi[n] * a;
        }
      }
      const double pn = nrm2(p, N);
      if (pn == 0.0) { degenerate = true; break; }                   // reading C7
      for (int64_t n = 0; n < N; ++n) p[n] /= pn;
      gemv_n(R, M, N, p, t);                                         // T^(k) <- R P^(k)
      for (int rep = 0; gs && k > 0 && rep < gs_passes; ++rep) {
        gemv_t(T, M, k, t, coef.data());                             // B <- V_(k)^T V^(k)
        for (int i = 0; i < k; ++i) {                                // V^(k) <- V^(k) - V_(k) B
          const double b = coef[i];
          const double* vi = T + id(0, i, M);
          for (int64_t m = 0; m < M; ++m) t[m] -= vi[m] * b;
        }
      }
      lam_new = nrm2(t, M);                                          // lambda' <- ||T^(k)||
      if (lam_new == 0.0) { degenerate = true; break; }              // reading C7
      if (gs)
        for (int64_t m = 0; m < M; ++m) t[m] /= lam_new;             // V^(k) <- V^(k)/lambda_k
      it = j + 1;
      if (test_mode == 0 ? (std::fabs(lam - lam_new) < eps * lam_new)  // PAPER.md:566,:1034 (C3)
                         : (std::fabs(lam_new - lam) <= eps)) break;   // PAPER.md:40,:84 (text)
      lam = lam_new;
    }
    if (degenerate) {
      for (int64_t m = 0; m < M; ++m) t[m] = 0.0;
      for (int64_t n = 0; n < N; ++n) p[n] = 0.0;
      lambda[k] = 0.0;
      iters[k] = 0;
      continue;                                                      // nothing to deflate
    }
    lambda[k] = lam_new;
    iters[k] = it;
    // R <- R - T^(k) P^(k)^T (eq. 3)  /  R <- R - lambda_k V^(k) U^(k)^T
    ger(R, M, N, gs ? -lam_new : -1.0, t, p);
  }
  if (gs)                                                            // T <- V Lambda
    for (int k = 0; k < K; ++k)
      for (int64_t m = 0; m < M; ++m) T[id(m, k, M)] *= lambda[k];
  if (R_out) std::memcpy(R_out, R, sizeof(double) * (size_t)M * (size_t)N);
  return 0;
}

int oracle_pca_ex(const double* X, int64_t M, int64_t N, int K, double eps, int max_iter, int algo, int test_mode,
                  double* T, double* P, double* lambda, int32_t* iters, double* R_out) {
  return oracle_pca_ex2(X, M, N, K, eps, max_iter, algo, test_mode, 1, T, P, lambda, iters, R_out);
}

int oracle_pca(const double* X, int64_t M, int64_t N, int K, double eps, int max_iter, int algo,
               double* T, double* P, double* lambda, int32_t* iters, double* R_out) {
  return oracle_pca_ex(X, M, N, K, eps, max_iter, algo, 0, T, P, lambda, iters, R_out);
}

// Cyclic Jacobi eigenvalue iteration for a real symmetric n x n matrix (textbook; Golub &
// Van Loan, "Matrix Computations", the paper's reference [Golub et al., 1996]).
//   A   in/out: n x n symmetric, col-major; destroyed (converges to diag(w))
//   w   out   : n eigenvalues (unsorted)
//   Vec out   : n x n, columns = eigenvectors, col-major
// Sweeps all (p,q) pairs until the off-diagonal Frobenius norm <= tol * ||A||_F or max_sweeps.
// returns number of sweeps used, or -1 on bad arguments.
int oracle_jacobi_eigh(double* A, int n, double* w, double* Vec, int max_sweeps, double tol) {
  if (!A || !w || !Vec || n < 1) return -1;
  for (int j = 0; j < n; ++j)
    for (int i = 0; i < n; ++i) Vec[id(i, j, n)] = (i == j) ? 1.0 : 0.0;
  double fro = 0.0;
  for (int64_t i = 0; i < (int64_t)n * n; ++i) fro += A[i] * A[i];
  fro = std::sqrt(fro);
  int sweep = 0;
  for (; sweep < max_sweeps; ++sweep) {
    double off = 0.0;
    for (int q = 0; q < n; ++q)
      for (int p = 0; p < n; ++p)
        if (p != q) off += A[id(p, q, n)] * A[id(p, q, n)];
    if (std::sqrt(off) <= tol * fro) break;
    for (int p = 0; p < n - 1; ++p) {
      for (int q = p + 1; q < n; ++q) {
        const double apq = A[id(p, q, n)];
        if (apq == 0.0) continue;
        const double app = A[id(p, p, n)], aqq = A[id(q, q, n)];
        const double theta = (aqq - app) / (2.0 * apq);
        const double tt = (theta >= 0.0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
        const double c = 1.0 / std::sqrt(tt * tt + 1.0), s = tt * c;
        for (int i = 0; i < n; ++i) {  // A <- A J  (columns p, q)
          const double aip = A[id(i, p, n)], aiq = A[id(i, q, n)];
          A[id(i, p, n)] = c * aip - s * aiq;
          A[id(i, q, n)] = s * aip + c * aiq;
        }
        for (int i = 0; i < n; ++i) {  // A <- J^T A  (rows p, q)
          const double api = A[id(p, i, n)], aqi = A[id(q, i, n)];
          A[id(p, i, n)] = c * api - s * aqi;
          A[id(q, i, n)] = s * api + c * aqi;
        }
        for (int i = 0; i < n; ++i) {  // Vec <- Vec J
          const double vip = Vec[id(i, p, n)], viq = Vec[id(i, q, n)];
          Vec[id(i, p, n)] = c * vip - s * viq;
          Vec[id(i, q, n)] = s * vip + c * viq;
        }
      }
    }
  }
  for (int i = 0; i < n; ++i) w[i] = A[id(i, i, n)];
  return sweep;
}

}  // extern "C"
