// K8: corner spectrum.  s = descending |eigenvalues| of the symmetric, Frobenius-
// normalised corner C (reading A6), delta = max_i |s_i - s_prev_i|.
//
// Algorithm (one CTA, chi <= a few hundred): Householder tridiagonalisation of a
// working copy W (lower triangle referenced, kept in global/L2), then every
// eigenvalue by Sturm-sequence bisection (one thread per eigenvalue), then a
// rank sort.  Bisection gives each eigenvalue to ~2 ulp of ||C|| = 1, which is
// what the convergence test (tol 1e-10..1e-12 absolute) needs.
#pragma once
#include "kernels_misc.cuh"

namespace qk {

// W: n x n working copy (destroyed).  dvec[n], evec[n] (evec[0] unused) out.
// scratch: vv[n], pv[n].
__global__ void tridiag_kernel(double* __restrict__ W, int n, double* __restrict__ dvec,
                               double* __restrict__ evec, double* __restrict__ vv, double* __restrict__ pv) {
  __shared__ double sh[33];
  __shared__ double s_tau, s_scale, s_beta;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  for (int k = 0; k < n - 2; ++k) {
    // reflector for column k, rows k+1..n-1
    double acc = 0.0;
    for (int i = k + 2 + tid; i < n; i += blockDim.x) {
      double x = W[(long long)i * n + k];
      acc = fma(x, x, acc);
    }
    double tail2 = block_sum(acc, sh);
    if (tid == 0) {
      double alpha = W[(long long)(k + 1) * n + k];
      double t = 0.0, scale = 0.0, beta = alpha;
      if (tail2 > 0.0) {
        double sigma = sqrt(fma(alpha, alpha, tail2));
        beta = alpha >= 0.0 ? -sigma : sigma;
        t = (beta - alpha) / beta;
        scale = 1.0 / (alpha - beta);
      }
      s_tau = t; s_scale = scale; s_beta = beta;
    }
    __syncthreads();
    const double tau = s_tau;
    if (tid == 0) { evec[k + 1] = s_beta; dvec[k] = W[(long long)k * n + k]; }
    if (tau == 0.0) { __syncthreads(); continue; }
    for (int i = k + 1 + tid; i < n; i += blockDim.x)
      vv[i] = (i == k + 1) ? 1.0 : W[(long long)i * n + k] * s_scale;
    __syncthreads();
    // p = tau * W22 v   (W22 symmetric; only the lower triangle is kept current)
    for (int i = k + 1 + warp; i < n; i += nwarp) {
      double a = 0.0;
      for (int j = k + 1 + lane; j < n; j += 32) {
        double wij = (j <= i) ? W[(long long)i * n + j] : W[(long long)j * n + i];
        a = fma(wij, vv[j], a);
      }
      a = warp_sum(a);
      if (lane == 0) pv[i] = tau * a;
    }
    __syncthreads();
    double acc2 = 0.0;
    for (int i = k + 1 + tid; i < n; i += blockDim.x) acc2 = fma(pv[i], vv[i], acc2);
    double pTv = block_sum(acc2, sh);
    double coef = 0.5 * tau * pTv;
    for (int i = k + 1 + tid; i < n; i += blockDim.x) pv[i] = fma(-coef, vv[i], pv[i]);   // w
    __syncthreads();
    // W22 <- W22 - v w^T - w v^T   (lower triangle)
    int nn = n - k - 1;
    for (long long idx = tid; idx < (long long)nn * nn; idx += blockDim.x) {
      int i = k + 1 + (int)(idx / nn), j = k + 1 + (int)(idx % nn);
      if (j <= i) {
        double x = W[(long long)i * n + j];
        x = fma(-vv[i], pv[j], x);
        x = fma(-pv[i], vv[j], x);
        W[(long long)i * n + j] = x;
      }
    }
    __syncthreads();
  }
  if (tid == 0) {
    if (n >= 2) {
      dvec[n - 2] = W[(long long)(n - 2) * n + (n - 2)];
      evec[n - 1] = W[(long long)(n - 1) * n + (n - 2)];
    }
    dvec[n - 1] = W[(long long)(n - 1) * n + (n - 1)];
    evec[0] = 0.0;
  }
}

// number of eigenvalues of the tridiagonal (d, e) that are < x
__device__ __forceinline__ int sturm_count(const double* d, const double* e2, int n, double x, double pivmin) {
  int cnt = 0;
  double q = d[0] - x;
  if (fabs(q) < pivmin) q = -pivmin;
  cnt += q < 0.0;
  for (int i = 1; i < n; ++i) {
    q = d[i] - x - e2[i] / q;
    if (fabs(q) < pivmin) q = -pivmin;
    cnt += q < 0.0;
  }
  return cnt;
}

// One block, blockDim.x >= n.  s_out: descending |lambda|; eig_out: signed eigenvalues
// ascending; delta_out[0] = max|s - s_prev|; then s_prev <- s (if update_prev).
__global__ void bisect_sort_kernel(const double* __restrict__ dvec, const double* __restrict__ evec, int n,
                                   double* __restrict__ eig_out, double* __restrict__ s_out,
                                   double* __restrict__ s_prev, double* __restrict__ delta_out, int update_prev) {
  extern __shared__ double shm[];          // d[n], e2[n], lam[n], red[33]
  double* d = shm; double* e2 = shm + n; double* lam = shm + 2 * n; double* red = shm + 3 * n;
  const int tid = threadIdx.x;
  double lo = INFINITY, hi = -INFINITY, emax = 0.0;
  for (int i = tid; i < n; i += blockDim.x) {
    d[i] = dvec[i];
    double e = i > 0 ? evec[i] : 0.0;
    e2[i] = e * e;
  }
  __syncthreads();
  for (int i = tid; i < n; i += blockDim.x) {
    double el = i > 0 ? sqrt(e2[i]) : 0.0, er = i + 1 < n ? sqrt(e2[i + 1]) : 0.0;
    lo = fmin(lo, d[i] - el - er);
    hi = fmax(hi, d[i] + el + er);
    emax = fmax(emax, e2[i]);
  }
  double ghi = block_max(hi, red);
  double glo = -block_max(-lo, red);
  double gemax = block_max(emax, red);
  double bnd = fmax(fabs(glo), fabs(ghi));
  double pivmin = fmax(2.2250738585072014e-308 * fmax(1.0, gemax), 1e-300);
  glo -= 2.0 * 2.220446049250313e-16 * bnd * n + 2.0 * pivmin;
  ghi += 2.0 * 2.220446049250313e-16 * bnd * n + 2.0 * pivmin;
  if (tid < n) {
    // eigenvalue number tid (ascending): smallest x with count(x) >= tid+1
    double a = glo, b = ghi;
    for (int it = 0; it < 200; ++it) {
      double mid = 0.5 * (a + b);
      if (mid <= a || mid >= b) break;
      if (sturm_count(d, e2, n, mid, pivmin) >= tid + 1) b = mid; else a = mid;
    }
    lam[tid] = 0.5 * (a + b);
  }
  __syncthreads();
  double dl = 0.0;
  if (tid < n) {
    double mine = fabs(lam[tid]);
    int rank = 0;
    for (int j = 0; j < n; ++j) {
      double o = fabs(lam[j]);
      rank += (o > mine) || (o == mine && j < tid);
    }
    eig_out[tid] = lam[tid];
    s_out[rank] = mine;
  }
  __syncthreads();
  if (tid < n) dl = fabs(s_out[tid] - s_prev[tid]);
  double dmax = block_max(dl, red);
  if (tid == 0) delta_out[0] = dmax;
  __syncthreads();
  if (update_prev && tid < n) s_prev[tid] = s_out[tid];
}

// ------------------------------------------------------------------------------
// Fast path (n(n+1)/2 doubles fit in one SM's shared memory, n <= ~236):
// the packed lower triangle L[i][j] (j <= i, offset i(i+1)/2 + j) lives in shared
// memory for the whole tridiagonalisation, so each Householder step costs shared-
// memory bandwidth instead of L2 round trips.  Same arithmetic as tridiag_kernel.
__device__ __forceinline__ int tri_off(int i) { return (i * (i + 1)) >> 1; }

__global__ void __launch_bounds__(1024, 1)
tridiag_smem_kernel(const double* __restrict__ Cmat, int n, double* __restrict__ dvec, double* __restrict__ evec) {
  extern __shared__ __align__(16) double tsm[];
  double* L = tsm;                              // n(n+1)/2
  double* vv = L + tri_off(n);                  // n
  double* pv = vv + n;                          // n
  double* sh = pv + n;                          // 33
  __shared__ double s_tau, s_scale, s_beta;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  for (int i = warp; i < n; i += nwarp)
    for (int j = lane; j <= i; j += 32) L[tri_off(i) + j] = Cmat[(long long)i * n + j];
  __syncthreads();
  for (int k = 0; k < n - 2; ++k) {
    double acc = 0.0;
    for (int i = k + 2 + tid; i < n; i += blockDim.x) {
      double x = L[tri_off(i) + k];
      acc = fma(x, x, acc);
    }
    double tail2 = block_sum(acc, sh);
    if (tid == 0) {
      double alpha = L[tri_off(k + 1) + k];
      double t = 0.0, scale = 0.0, beta = alpha;
      if (tail2 > 0.0) {
        double sigma = sqrt(fma(alpha, alpha, tail2));
        beta = alpha >= 0.0 ? -sigma : sigma;
        t = (beta - alpha) / beta;
        scale = 1.0 / (alpha - beta);
      }
      s_tau = t; s_scale = scale; s_beta = beta;
      evec[k + 1] = beta; dvec[k] = L[tri_off(k) + k];
    }
    __syncthreads();
    const double tau = s_tau;
    if (tau == 0.0) { __syncthreads(); continue; }
    for (int i = k + 1 + tid; i < n; i += blockDim.x) vv[i] = (i == k + 1) ? 1.0 : L[tri_off(i) + k] * s_scale;
    __syncthreads();
    for (int i = k + 1 + warp; i < n; i += nwarp) {            // p = tau * W22 v
      double a = 0.0;
      const double* Li = L + tri_off(i);
      for (int j = k + 1 + lane; j < n; j += 32) {
        double wij = (j <= i) ? Li[j] : L[tri_off(j) + i];
        a = fma(wij, vv[j], a);
      }
      a = warp_sum(a);
      if (lane == 0) pv[i] = tau * a;
    }
    __syncthreads();
    double acc2 = 0.0;
    for (int i = k + 1 + tid; i < n; i += blockDim.x) acc2 = fma(pv[i], vv[i], acc2);
    double pTv = block_sum(acc2, sh);
    double coef = 0.5 * tau * pTv;
    __syncthreads();
    for (int i = k + 1 + tid; i < n; i += blockDim.x) pv[i] = fma(-coef, vv[i], pv[i]);   // w
    __syncthreads();
    for (int i = k + 1 + warp; i < n; i += nwarp) {            // W22 -= v w^T + w v^T (lower triangle)
      double* Li = L + tri_off(i);
      const double vi = vv[i], wi = pv[i];
      for (int j = k + 1 + lane; j <= i; j += 32) {
        double x = Li[j];
        x = fma(-vi, pv[j], x);
        x = fma(-wi, vv[j], x);
        Li[j] = x;
      }
    }
    __syncthreads();
  }
  if (tid == 0) {
    if (n >= 2) {
      dvec[n - 2] = L[tri_off(n - 2) + n - 2];
      evec[n - 1] = L[tri_off(n - 1) + n - 2];
    }
    dvec[n - 1] = L[tri_off(n - 1) + n - 1];
    evec[0] = 0.0;
  }
}

// Eigenvalues of the tridiagonal by warp-multisection: warp w of block B finds
// eigenvalue number idx = 8 B + w (ascending; see `ke` for the partial mode).  Each iteration the 32 lanes evaluate
// the Sturm count at 32 interior points of [a, b], shrinking the bracket 33-fold
// (about 11 iterations to the last ulp instead of ~55 bisection steps).
__global__ void __launch_bounds__(256)
multisect_kernel(const double* __restrict__ dvec, const double* __restrict__ evec, int n,
                 double* __restrict__ eig_out, int ke = 0) {
  extern __shared__ double msm[];               // d[n], e2[n], red[33]
  double* d = msm; double* e2 = msm + n; double* red = msm + 2 * n;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int i = tid; i < n; i += blockDim.x) {
    d[i] = dvec[i];
    double e = i > 0 ? evec[i] : 0.0;
    e2[i] = e * e;
  }
  __syncthreads();
  double lo = INFINITY, hi = -INFINITY, emax = 0.0;
  for (int i = tid; i < n; i += blockDim.x) {
    double el = i > 0 ? sqrt(e2[i]) : 0.0, er = i + 1 < n ? sqrt(e2[i + 1]) : 0.0;
    lo = fmin(lo, d[i] - el - er);
    hi = fmax(hi, d[i] + el + er);
    emax = fmax(emax, e2[i]);
  }
  double ghi = block_max(hi, red);
  double glo = -block_max(-lo, red);
  double gemax = block_max(emax, red);
  const double bnd = fmax(fabs(glo), fabs(ghi));
  const double pivmin = fmax(2.2250738585072014e-308 * fmax(1.0, gemax), 1e-300);
  glo -= 2.0 * 2.220446049250313e-16 * bnd * n + 2.0 * pivmin;
  ghi += 2.0 * 2.220446049250313e-16 * bnd * n + 2.0 * pivmin;
  // ke > 0 (and 2 ke < n): only the ke smallest and the ke largest eigenvalues, written compactly
  // (slot c < ke: eigenvalue c; slot c >= ke: eigenvalue n - 2 ke + c) -- the eigen step's candidates.
  const int slot = blockIdx.x * 8 + warp;
  const bool part = ke > 0 && 2 * ke < n;
  if (slot >= (part ? 2 * ke : n)) return;
  const int idx = (part && slot >= ke) ? n - 2 * ke + slot : slot;
  double a = glo, b = ghi;
  for (int it = 0; it < 64; ++it) {
    const double h = (b - a) / 33.0;
    const double x = a + (lane + 1) * h;
    const bool inside = x > a && x < b;
    int cnt = inside ? sturm_count(d, e2, n, x, pivmin) : (x >= b ? n : 0);
    const unsigned m = __ballot_sync(0xffffffffu, cnt >= idx + 1);
    const int f = m ? __ffs(m) - 1 : 32;                       // first point with count >= idx+1
    const double xb = __shfl_sync(0xffffffffu, x, f < 32 ? f : 31);
    const double xa = __shfl_sync(0xffffffffu, x, f > 0 ? f - 1 : 0);
    const double nb = f < 32 ? fmin(xb, b) : b;
    const double na = f > 0 ? fmax(xa, a) : a;
    const bool progress = (nb < b) || (na > a);
    a = na; b = nb;
    if (!progress || !(b - a > 0.0)) break;
  }
  if (lane == 0) eig_out[slot] = 0.5 * (a + b);
}

// One block, blockDim.x >= n: s = sorted |eig| (descending), delta vs s_prev.
__global__ void spectrum_finalize_kernel(const double* __restrict__ eig, int n, double* __restrict__ s_out,
                                         double* __restrict__ s_prev, double* __restrict__ delta_out,
                                         int update_prev) {
  extern __shared__ double fsm[];               // lam[n], red[33]
  double* lam = fsm; double* red = fsm + n;
  const int tid = threadIdx.x;
  if (tid < n) lam[tid] = eig[tid];
  __syncthreads();
  if (tid < n) {
    double mine = fabs(lam[tid]);
    int rank = 0;
    for (int j = 0; j < n; ++j) {
      double o = fabs(lam[j]);
      rank += (o > mine) || (o == mine && j < tid);
    }
    s_out[rank] = mine;
  }
  __syncthreads();
  double dl = 0.0;
  if (tid < n) dl = fabs(s_out[tid] - s_prev[tid]);
  double dmax = block_max(dl, red);
  if (tid == 0) delta_out[0] = dmax;
  __syncthreads();
  if (update_prev && tid < n) s_prev[tid] = s_out[tid];
}

}  // namespace qk
