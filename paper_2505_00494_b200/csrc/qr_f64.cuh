// K2: unpivoted Householder QR of the reduced corner c~ (rows x n, row-major,
// ld = n).  Reflector convention (LAPACK dlarfg): for a column x
// with head alpha and tail t:  sigma = ||x||, beta = -sign(alpha) sigma,
// tau = (beta - alpha)/beta, v = [1; t/(alpha - beta)], H = I - tau v v^T,
// H x = beta e_1.  R's diagonal is beta; the later sign fix makes it >= 0.
//
// Level-2 column kernels (this file, first section) are the simple correct path;
// the blocked compact-WY path (second section) uses them only inside a panel.
#pragma once
#include "kernels_misc.cuh"

namespace qk {

// One block.  Column k of X (rows k..rows-1): compute the reflector in place.
// X[k,k] <- beta, X[i>k,k] <- v_i, tau[k] <- tau.
__global__ void house_col_kernel(double* __restrict__ X, long long ld, long long rows, int k,
                                 double* __restrict__ tau) {
  __shared__ double sh[33];
  __shared__ double s_scale;
  // scaled 2-norm is unnecessary here: entries are O(1) after normalisation of C, T
  double acc = 0.0;
  for (long long i = k + 1 + threadIdx.x; i < rows; i += blockDim.x) {
    double v = X[i * ld + k];
    acc = fma(v, v, acc);
  }
  double tail2 = block_sum(acc, sh);
  if (threadIdx.x == 0) {
    double alpha = X[(long long)k * ld + k];
    double t = 0.0, scale = 0.0, beta = alpha;
    if (tail2 > 0.0) {
      double sigma = sqrt(fma(alpha, alpha, tail2));
      beta = alpha >= 0.0 ? -sigma : sigma;
      t = (beta - alpha) / beta;
      scale = 1.0 / (alpha - beta);
    }
    tau[k] = t;
    s_scale = scale;
    X[(long long)k * ld + k] = beta;
  }
  __syncthreads();
  double scale = s_scale;
  for (long long i = k + 1 + threadIdx.x; i < rows; i += blockDim.x) X[i * ld + k] *= scale;
}

// Apply H_k = I - tau v v^T (v stored in column k of V below the diagonal, v_k = 1)
// to columns [c0, c1) of Y, rows k..rows-1.  Each block owns CPB columns.
template <int CPB>
__global__ void house_apply_kernel(const double* __restrict__ V, long long ldv, long long rows, int k,
                                   const double* __restrict__ tau, double* __restrict__ Y, long long ldy,
                                   int c0, int c1) {
  __shared__ double sh[33];
  __shared__ double w[CPB];
  const double t = tau[k];
  if (t == 0.0) return;
  int cb = c0 + blockIdx.x * CPB;
  double acc[CPB];
#pragma unroll
  for (int c = 0; c < CPB; ++c) acc[c] = 0.0;
  for (long long i = k + threadIdx.x; i < rows; i += blockDim.x) {
    double v = (i == k) ? 1.0 : V[i * ldv + k];
#pragma unroll
    for (int c = 0; c < CPB; ++c)
      if (cb + c < c1) acc[c] = fma(v, Y[i * ldy + cb + c], acc[c]);
  }
#pragma unroll
  for (int c = 0; c < CPB; ++c) {
    double s = block_sum(acc[c], sh);
    if (threadIdx.x == 0) w[c] = t * s;
  }
  __syncthreads();
  for (long long i = k + threadIdx.x; i < rows; i += blockDim.x) {
    double v = (i == k) ? 1.0 : V[i * ldv + k];
#pragma unroll
    for (int c = 0; c < CPB; ++c)
      if (cb + c < c1) Y[i * ldy + cb + c] = fma(-v, w[c], Y[i * ldy + cb + c]);
  }
}

}  // namespace qk
