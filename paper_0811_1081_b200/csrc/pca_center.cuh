// =====================================================================================
// pca_center.cuh -- step S0, mean centring (eq. 1 / PAPER.md:21-23), in place.
//
// Default (reading C1, "each column is mean centered", columns = attributes):
//   mu_n = (1/M) sum_m X[m,n];  X[m,n] -= mu_n
// One CTA per column (grid-stride over columns).  The column is read once from HBM to form the
// mean in fp64, then re-read (L2-hot: a column is at most a few hundred KB) and written back, so
// DRAM traffic is one read + one write of X.  The paper does this with 2N level-1 BLAS launches
// (PAPER.md:1009-1013).
//
// Literal eq. (1) mode: the mean COLUMN U/N, U = sum_n X^(n), is subtracted from every column,
// i.e. every row loses its mean over the N columns (listing PAPER.md:1009-1013).
// =====================================================================================
#pragma once
#include "pca_device.cuh"

namespace pca {

constexpr int kCenterThreads = 512;

__global__ void __launch_bounds__(kCenterThreads) pca_center_columns_kernel(float* __restrict__ X, long long M, int N,
                                                                            int vec4) {
  __shared__ double red[kCenterThreads / 32 + 1];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  for (int n = blockIdx.x; n < N; n += gridDim.x) {
    float* col = X + (size_t)n * M;
    double s = 0.0;
    if (vec4) {
      const long long m4 = M >> 2;
      for (long long i = tid; i < m4; i += kCenterThreads) {
        const float4 v = __ldcg(reinterpret_cast<const float4*>(col) + i);
        s += ((double)v.x + (double)v.y) + ((double)v.z + (double)v.w);
      }
    } else {
      for (long long i = tid; i < M; i += kCenterThreads) s += (double)__ldcg(col + i);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    __syncthreads();
    if (lane == 0) red[w] = s;
    __syncthreads();
    if (w == 0) {
      double t = (lane < kCenterThreads / 32) ? red[lane] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
      if (lane == 0) red[kCenterThreads / 32] = t / (double)M;
    }
    __syncthreads();
    const double mu = red[kCenterThreads / 32];
    if (vec4) {
      const long long m4 = M >> 2;
      for (long long i = tid; i < m4; i += kCenterThreads) {
        float4 v = __ldcg(reinterpret_cast<const float4*>(col) + i);
        v.x = (float)((double)v.x - mu);
        v.y = (float)((double)v.y - mu);
        v.z = (float)((double)v.z - mu);
        v.w = (float)((double)v.w - mu);
        reinterpret_cast<float4*>(col)[i] = v;
      }
    } else {
      for (long long i = tid; i < M; i += kCenterThreads) col[i] = (float)((double)__ldcg(col + i) - mu);
    }
  }
}

// Literal eq. (1): thread per row, coalesced across rows, loop over the N columns twice.
__global__ void __launch_bounds__(256) pca_center_eq1_kernel(float* __restrict__ X, long long M, int N) {
  const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= M) return;
  double u = 0.0;
  for (int n = 0; n < N; ++n) u += (double)__ldcg(X + (size_t)n * M + m);
  const double mean = u / (double)N;
  for (int n = 0; n < N; ++n) {
    float* p = X + (size_t)n * M + m;
    *p = (float)((double)__ldcg(p) - mean);
  }
}

// fp64 storage (the paper's precision): same two kernels on double data
__global__ void __launch_bounds__(kCenterThreads) pca_center_columns_f64_kernel(double* __restrict__ X, long long M, int N) {
  __shared__ double red[kCenterThreads / 32 + 1];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  for (int n = blockIdx.x; n < N; n += gridDim.x) {
    double* col = X + (size_t)n * M;
    double s = 0.0;
    for (long long i = tid; i < M; i += kCenterThreads) s += __ldcg(col + i);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    __syncthreads();
    if (lane == 0) red[w] = s;
    __syncthreads();
    if (w == 0) {
      double t = (lane < kCenterThreads / 32) ? red[lane] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
      if (lane == 0) red[kCenterThreads / 32] = t / (double)M;
    }
    __syncthreads();
    const double mu = red[kCenterThreads / 32];
    for (long long i = tid; i < M; i += kCenterThreads) col[i] = __ldcg(col + i) - mu;
  }
}

__global__ void __launch_bounds__(256) pca_center_eq1_f64_kernel(double* __restrict__ X, long long M, int N) {
  const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= M) return;
  double u = 0.0;
  for (int n = 0; n < N; ++n) u += __ldcg(X + (size_t)n * M + m);
  const double mean = u / (double)N;
  for (int n = 0; n < N; ++n) {
    double* p = X + (size_t)n * M + m;
    *p = __ldcg(p) - mean;
  }
}

}  // namespace pca
