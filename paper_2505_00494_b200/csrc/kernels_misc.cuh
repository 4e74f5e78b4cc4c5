// Bandwidth-/latency-bound kernels of the QR-CTMRG step: K0 (a-builder), K7
// (symmetrise + Frobenius-normalise), K8 (corner spectrum), sign fix, helpers.
// All reductions use fixed trees (deterministic; no floating-point atomics).
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace qk {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
// Block-wide sum, result valid in every thread.  blockDim.x multiple of 32, <= 1024.
__device__ __forceinline__ double block_sum(double v, double* sh /* >= 33 doubles */) {
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  v = warp_sum(v);
  __syncthreads();
  if (lane == 0) sh[w] = v;
  __syncthreads();
  if (w == 0) {
    double t = lane < nw ? sh[lane] : 0.0;
    t = warp_sum(t);
    if (lane == 0) sh[32] = t;
  }
  __syncthreads();
  return sh[32];
}
__device__ __forceinline__ double block_max(double v, double* sh) {
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  v = warp_max(v);
  __syncthreads();
  if (lane == 0) sh[w] = v;
  __syncthreads();
  if (w == 0) {
    double t = lane < nw ? sh[lane] : -INFINITY;
    t = warp_max(t);
    if (lane == 0) sh[32] = t;
  }
  __syncthreads();
  return sh[32];
}

// ---------------------------------------------------------------- K0: (E0)
// a[(u u'),(l l'),(d d'),(r r')] = sum_s A[s,u,l,d,r] A[s,u',l',d',r']
// written as the K x N matrix a_mat[(u,l)][(d,r)] with leading dimension lda_a
// (padded so every row is 16-byte aligned for the GEMM's vector loads).
__global__ void build_a_kernel(const double* __restrict__ A, int d, int D, double* __restrict__ a_mat,
                               long long lda_a) {
  // one block per matrix row (u,l); threads run along the contiguous column index (d,r)
  const int b = D * D, b2 = b * b;
  const long long DD = (long long)D * D * D * D;
  const int row = blockIdx.x, u = row / b, l = row % b;
  const int uk = u / D, ub = u % D, lk = l / D, lb = l % D;
  const long long rk0 = ((long long)uk * D + lk) * D * D, rb0 = ((long long)ub * D + lb) * D * D;
  double* out = a_mat + (long long)row * lda_a;
  for (int c = threadIdx.x; c < b2; c += blockDim.x) {
    const int dd = c / b, r = c % b;
    const int dk = dd / D, db = dd % D, rk = r / D, rb = r % D;
    const long long ik = rk0 + dk * D + rk, ib = rb0 + db * D + rb;
    double s = 0.0;
    for (int sidx = 0; sidx < d; ++sidx) s = fma(A[sidx * DD + ik], A[sidx * DD + ib], s);
    out[c] = s;
  }
}

// a^{s s'}[(u u'),(l l'),(d d'),(r r')] = A[s,u,l,d,r] A[s',u',l',d',r']  (physical legs open; NEXT-3 energy),
// same K x N matrix layout as build_a_kernel.
__global__ void build_a_pair_kernel(const double* __restrict__ A, int D, int s, int sp, double* __restrict__ a_mat,
                                    long long lda_a) {
  const int b = D * D;
  const long long n = (long long)b * b * b * b;
  const long long DD = (long long)D * D * D * D;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    int r = (int)(idx % b), dd = (int)((idx / b) % b), l = (int)((idx / ((long long)b * b)) % b),
        u = (int)(idx / ((long long)b * b * b));
    int uk = u / D, ub = u % D, lk = l / D, lb = l % D, dk = dd / D, db = dd % D, rk = r / D, rb = r % D;
    long long ik = (((long long)uk * D + lk) * D + dk) * D + rk;
    long long ib = (((long long)ub * D + lb) * D + db) * D + rb;
    a_mat[((long long)u * b + l) * lda_a + (long long)dd * b + r] = A[s * DD + ik] * A[sp * DD + ib];
  }
}

// Re-laid-out copies of A for the layered absorption (NEXT-1):
//   B1[(u_k,l_k)][(s,d_k,r_k)] = A[s,u_k,l_k,d_k,r_k]   (D^2 x d D^2, leading dimension ld1)
//   B2[(s,u_b,l_b)][(d_b,r_b)] = A[s,u_b,l_b,d_b,r_b]   (d D^2 x D^2, leading dimension ld2)
__global__ void build_layers_kernel(const double* __restrict__ A, int d, int D, double* __restrict__ B1,
                                    long long ld1, double* __restrict__ B2, long long ld2) {
  const long long n = (long long)d * D * D * D * D;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    int r = (int)(idx % D), dd = (int)((idx / D) % D), l = (int)((idx / (D * D)) % D),
        u = (int)((idx / ((long long)D * D * D)) % D), sidx = (int)(idx / ((long long)D * D * D * D));
    const double v = A[idx];
    B1[((long long)u * D + l) * ld1 + ((long long)sidx * D + dd) * D + r] = v;
    B2[(((long long)sidx * D + u) * D + l) * ld2 + (long long)dd * D + r] = v;
  }
}

// ---------------------------------------------------------------- K7
// Pass 1: dst = sym(src) (or copy), per-block partial sums of squares in a fixed
// order.  C part: n x n matrix.  T part: (chi, b, chi) swapping the chi legs.
// Blocks [0, nbC) handle C, blocks [nbC, nbC+nbT) handle T.
__global__ void sym_partial_kernel(const double* __restrict__ Cn, const double* __restrict__ Tn, int chi, int b,
                                   int symmetrize, double* __restrict__ C, double* __restrict__ T,
                                   double* __restrict__ partial, int nbC, int nbT) {
  __shared__ double sh[33];
  double acc = 0.0;
  if ((int)blockIdx.x < nbC) {
    long long n = (long long)chi * chi;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
         idx += (long long)nbC * blockDim.x) {
      int i = (int)(idx / chi), j = (int)(idx % chi);
      double v = Cn[idx];
      if (symmetrize) v = 0.5 * (v + Cn[(long long)j * chi + i]);
      C[idx] = v;
      acc = fma(v, v, acc);
    }
  } else {
    int blk = blockIdx.x - nbC;
    long long n = (long long)chi * b * chi, bc = (long long)b * chi;
    for (long long idx = (long long)blk * blockDim.x + threadIdx.x; idx < n; idx += (long long)nbT * blockDim.x) {
      int i = (int)(idx / bc), s = (int)((idx / chi) % b), k = (int)(idx % chi);
      double v = Tn[idx];
      if (symmetrize) v = 0.5 * (v + Tn[(long long)k * bc + (long long)s * chi + i]);
      T[idx] = v;
      acc = fma(v, v, acc);
    }
  }
  double tot = block_sum(acc, sh);
  if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

// Pass 2: every block re-reduces the partials in the same fixed order, then scales.
// scal[0] = ||C||_F, scal[1] = ||T||_F ; flag set to 1 on NaN/Inf/zero norm.
// hist != null: this K7 closes an iteration; block 0 appends the record {delta = NaN (filled in by K8 if the step is
// checked), ||C'||_F, ||T'||_F, min_k R_kk / max_k R_kk} to the ring buffer hist[QRCTM_HIST_CAP][4] and bumps *hist_n.
constexpr int QRCTM_HIST_CAP = 4096;
__global__ void scale_kernel(double* __restrict__ C, double* __restrict__ T, int chi, int b,
                             const double* __restrict__ partial, int nbC, int nbT, double* __restrict__ scal,
                             int* __restrict__ flag, double* __restrict__ hist = nullptr, int* __restrict__ hist_n = nullptr,
                             const double* __restrict__ R = nullptr) {
  __shared__ double sh[33];
  if (hist && blockIdx.x == 0) {
    double mn = INFINITY, mx = -INFINITY;
    for (int k = threadIdx.x; k < chi; k += blockDim.x) { const double v = R[(long long)k * chi + k]; mn = fmin(mn, v); mx = fmax(mx, v); }
    const double gmx = block_max(mx, sh);
    const double gmn = -block_max(-mn, sh);
    if (threadIdx.x == 0) scal[8] = gmx != 0.0 ? gmn / gmx : 0.0;
  }
  double a = 0.0, t = 0.0;
  for (int i = threadIdx.x; i < nbC; i += blockDim.x) a += partial[i];
  for (int i = threadIdx.x; i < nbT; i += blockDim.x) t += partial[nbC + i];
  double sc = block_sum(a, sh);
  double st = block_sum(t, sh);
  double nc = sqrt(sc), nt = sqrt(st);
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    scal[0] = nc; scal[1] = nt;
    if (!(nc > 0.0) || !(nt > 0.0) || isinf(nc) || isinf(nt)) *flag = 1;
    if (hist) {
      const int idx = *hist_n;
      double* rec = hist + (size_t)(idx % QRCTM_HIST_CAP) * 4;
      rec[0] = __longlong_as_double(0x7ff8000000000000LL); rec[1] = nc; rec[2] = nt; rec[3] = scal[8];
      *hist_n = idx + 1;
    }
  }
  double ic = 1.0 / nc, it = 1.0 / nt;
  long long n1 = (long long)chi * chi, n2 = (long long)chi * b * chi;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n1 + n2;
       idx += (long long)gridDim.x * blockDim.x) {
    if (idx < n1) C[idx] = C[idx] / nc;
    else T[idx - n1] = T[idx - n1] / nt;
  }
  (void)ic; (void)it;
}

// ---------------------------------------------------------------- sign fix (A7)
// s_k = -1 if R_kk < 0 else +1 ;  R[k,:] *= s_k ; Q[:,k] *= s_k.  Also zeroes R below the diagonal.
__global__ void sign_fix_kernel(double* __restrict__ Q, long long rows, int n, double* __restrict__ R) {
  long long total = rows * n + (long long)n * n;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (long long)gridDim.x * blockDim.x) {
    if (idx < rows * n) {
      int k = (int)(idx % n);
      if (R[(long long)k * n + k] < 0.0) Q[idx] = -Q[idx];
    }
  }
}
__global__ void sign_fix_R_kernel(double* __restrict__ R, int n) {
  // one block per row k (run AFTER sign_fix_kernel has read the diagonal)
  int k = blockIdx.x;
  __shared__ double dk;
  if (threadIdx.x == 0) dk = R[(long long)k * n + k];
  __syncthreads();
  double s = dk < 0.0 ? -1.0 : 1.0;
  for (int j = threadIdx.x; j < n; j += blockDim.x) {
    double v = R[(long long)k * n + j];
    R[(long long)k * n + j] = j < k ? 0.0 : s * v;
  }
}

// ---------------------------------------------------------------- small helpers
__global__ void set_identity_top_kernel(double* __restrict__ Q, long long rows, int n) {
  long long total = rows * n;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (long long)gridDim.x * blockDim.x) {
    long long i = idx / n; int j = (int)(idx % n);
    Q[idx] = (i == j) ? 1.0 : 0.0;
  }
}
__global__ void copy_triu_kernel(const double* __restrict__ X, long long ldx, int n, double* __restrict__ R) {
  for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n * n; idx += gridDim.x * blockDim.x) {
    int i = idx / n, j = idx % n;
    R[idx] = j >= i ? X[(long long)i * ldx + j] : 0.0;
  }
}
__global__ void transpose_small_kernel(const double* __restrict__ Rm, int n, double* __restrict__ Rt) {
  for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n * n; idx += gridDim.x * blockDim.x) {
    int i = idx / n, j = idx % n;
    Rt[(long long)j * n + i] = Rm[idx];
  }
}
// NEXT-4 helpers: a column slice of a row-major matrix made contiguous, and the transposed row slice of R.
//   dst[i][c] = src[i][c0 + c] for c < nc, 0 for nc <= c < ldd   (rows x ldd, src leading dimension ld)
__global__ void slice_cols_kernel(const double* __restrict__ src, long long rows, int ld, int c0, int nc, int ldd,
                                  double* __restrict__ dst) {
  const long long total = rows * ldd;
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
       idx += (long long)gridDim.x * blockDim.x) {
    const long long i = idx / ldd; const int c = (int)(idx % ldd);
    dst[idx] = c < nc ? src[i * ld + c0 + c] : 0.0;
  }
}
//   Rt[k][r] = Rm[r0 + r][k] for r < nr, 0 for nr <= r < ldt     (n x ldt)
__global__ void transpose_rows_kernel(const double* __restrict__ Rm, int n, int r0, int nr, int ldt,
                                      double* __restrict__ Rt) {
  for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n * ldt; idx += gridDim.x * blockDim.x) {
    const int k = idx / ldt, r = idx % ldt;
    Rt[idx] = r < nr ? Rm[(long long)(r0 + r) * n + k] : 0.0;
  }
}
// dot of two arrays with a fixed tree: partial per block, then final by block 0 of a 2nd launch
__global__ void dot_partial_kernel(const double* __restrict__ x, const double* __restrict__ y, long long n,
                                   double* __restrict__ partial) {
  __shared__ double sh[33];
  double acc = 0.0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    acc = fma(x[i], y[i], acc);
  double t = block_sum(acc, sh);
  if (threadIdx.x == 0) partial[blockIdx.x] = t;
}
__global__ void sum_partial_kernel(const double* __restrict__ partial, int n, double* __restrict__ out) {
  __shared__ double sh[33];
  double a = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) a += partial[i];
  double t = block_sum(a, sh);
  if (threadIdx.x == 0) *out = t;
}
// trace(M*M) for a symmetric n x n matrix M == sum of squares; here generic: tr(M @ M) = sum_ij M_ij M_ji
__global__ void trace_prod_partial_kernel(const double* __restrict__ M, int n, double* __restrict__ partial) {
  __shared__ double sh[33];
  double acc = 0.0;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < (long long)n * n;
       idx += (long long)gridDim.x * blockDim.x) {
    int i = (int)(idx / n), j = (int)(idx % n);
    acc = fma(M[idx], M[(long long)j * n + i], acc);
  }
  double t = block_sum(acc, sh);
  if (threadIdx.x == 0) partial[blockIdx.x] = t;
}

}  // namespace qk
