// NEXT-2: the standard (eigen) CTMRG step needs "the chi eigenvectors with the largest
// magnitudes" of the symmetric enlarged corner C~ (reading A9).
// Hand-written symmetric eigensolver for the k largest-|lambda| pairs of an n x n matrix:
//   1. Householder tridiagonalisation, one reflector per step, all SMs:
//        eigh_reflector_kernel (one CTA)  : finishes w_{k-1}, brings row k up to date, builds v_k
//        eigh_pass_kernel      (grid)     : applies the pending rank-2 update of reflector k-1 to the upper
//                                           triangle of the trailing block and, in the same sweep, the
//                                           row and column partial sums of y = A22 v_k
//        eigh_ysum_kernel      (grid)     : y from the partials, fixed order
//      (one read + one write of HALF the trailing block per step; HBM/L2-bound)
//   2. the k smallest and k largest eigenvalues of the tridiagonal by warp multisection (spectrum.cuh)
//   3. eigh_select_kernel: the k of largest magnitude, stable in ascending-eigenvalue order
//   4. eigh_invit_kernel: inverse iteration on the tridiagonal, one thread per vector,
//      partial-pivoting LU recomputed each sweep, random start vectors
//   5. Householder QR of the n x k vectors (qr_f64.cuh) -- orthonormality to rounding even for
//      clustered eigenvalues; R's positive diagonal keeps every vector's direction
//   6. eigh_backtransform_kernel: U = H_0 ... H_{n-3} Z, two columns per CTA held in shared memory
//   7. eigh_sign_kernel: largest-|.| component of every column made positive (the sign gauge DESIGN.md fixes)
#pragma once
#include "kernels_misc.cuh"

namespace qk {

constexpr int EIGH_CW = 256;      // columns per chunk of the tridiagonalisation sweep

// First statement of the three tridiagonalisation kernels (launched with programmatic stream serialisation): let the
// next kernel in the stream be set up now, then wait until the previous one has completed and flushed its writes.
__device__ __forceinline__ void eigh_pdl_sync() {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
}

// sum_{t = t0}^{t1 - 1} part[t * stride], added in index order; loads issued eight at a time (the plain loop
// would wait for every load before issuing the next)
__device__ __forceinline__ double eigh_strided_sum(const double* __restrict__ part, long long stride, int t0, int t1,
                                                   double acc) {
  int t = t0;
  for (; t + 8 <= t1; t += 8) {
    double v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = part[(long long)(t + u) * stride];
#pragma unroll
    for (int u = 0; u < 8; ++u) acc += v[u];
  }
  for (; t < t1; ++t) acc += part[(long long)t * stride];
  return acc;
}

// One CTA.  Step k of the tridiagonalisation of W (n x n, row-major, symmetric; rows/cols >= k live).
//   k > 0 : y = A22 v_{k-1} (rows k..n-1, from eigh_ysum_kernel, or summed here when rg_prev > 0); forms w_{k-1} = p - (tau/2)(p.v) v, p = tau y
//   row k brought up to date: r[j] = W[k][j] - v[k] w[j] - w[k] v[j]  (j >= k)
//   k <= n-3: reflector v_k from r[k+1..], stored in vnew[] and in W[k][k+2..] (v_k[k+1] = 1 implied)
//   k == n-2: the last 2x2 block: d[n-2], e[n-1], d[n-1]
// Reflector convention as in K2 (LAPACK dlarfg): beta = -sign(alpha) ||x||, tau = (beta-alpha)/beta.
// Thread t owns columns k + t, k + t + 1024, ... (RMAX of them, n - k <= 1024 RMAX) in registers through all phases.
template <int RMAX>
__global__ void __launch_bounds__(1024, 1)
eigh_reflector_kernel(double* __restrict__ W, int n, int k, const double* __restrict__ y,
                      const double* __restrict__ rowpart, const double* __restrict__ colpart, int rg_prev,
                      const double* __restrict__ vprev, double* __restrict__ wv, double* __restrict__ vnew,
                      double* __restrict__ tauv, double* __restrict__ dvec, double* __restrict__ evec) {
  __shared__ double sh[33];
  __shared__ double s_vk, s_wk, s_alpha;
  eigh_pdl_sync();
  const int tid = threadIdx.x;
  double* Wk = W + (long long)k * n;
  double vp[RMAX], x[RMAX];              // v_{k-1}[i];  w_{k-1}[i], then the updated row entry r[i]
  const bool pending = k > 0;
  if (pending) {
    const double tau = tauv[k - 1];
    double acc = 0.0;
#pragma unroll
    for (int r = 0; r < RMAX; ++r) {
      const int i = k + tid + 1024 * r;
      double yi = 0.0; vp[r] = 0.0;
      if (i < n) {
        if (rg_prev > 0) {          // short tail: sum the sweep's partials here (same order as eigh_ysum_kernel)
          const int ii = i - k, nch = (n - k + EIGH_CW - 1) / EIGH_CW;
          yi = eigh_strided_sum(rowpart + i, n, ii / EIGH_CW, nch, yi);
          yi = eigh_strided_sum(colpart + i, n, 0, ii / rg_prev + 1, yi);
        } else {
          yi = y[i];
        }
        vp[r] = vprev[i];
      }
      x[r] = tau * yi;
      acc = fma(x[r], vp[r], acc);
    }
    const double pTv = block_sum(acc, sh);
    const double coef = 0.5 * tau * pTv;
#pragma unroll
    for (int r = 0; r < RMAX; ++r) {
      const int i = k + tid + 1024 * r;
      x[r] = fma(-coef, vp[r], x[r]);
      if (i < n) wv[i] = x[r];
    }
    if (tid == 0) { s_vk = vp[0]; s_wk = x[0]; }
    __syncthreads();
  }
  const double vk = pending ? s_vk : 0.0, wk = pending ? s_wk : 0.0;
  double acc = 0.0, d1 = 0.0;
#pragma unroll
  for (int r = 0; r < RMAX; ++r) {
    const int i = k + tid + 1024 * r;
    double xi = i < n ? Wk[i] : 0.0;
    if (pending) {
      if (i == k + 1) d1 = -2.0 * vp[r] * x[r];        // correction of W[k+1][k+1] (final block only)
      xi = fma(-vk, x[r], xi); xi = fma(-wk, vp[r], xi);
    }
    x[r] = xi;
    if (i >= k + 2) acc = fma(xi, xi, acc);
  }
  if (tid == 1 && k + 1 < n) s_alpha = x[0];
  if (k >= n - 2) {            // final block (n >= 2: k = n-2; n == 1: k = 0)
    if (tid == 0) { dvec[k] = x[0]; evec[0] = 0.0; }
    if (tid == 1 && k + 1 < n) { evec[k + 1] = x[0]; dvec[k + 1] = W[(long long)(k + 1) * n + (k + 1)] + d1; }
    return;
  }
  const double tail2 = block_sum(acc, sh);
  const double alpha = s_alpha;
  double t = 0.0, scale = 0.0, beta = alpha;
  if (tail2 > 0.0) {
    const double sigma = sqrt(fma(alpha, alpha, tail2));
    beta = alpha >= 0.0 ? -sigma : sigma;
    t = (beta - alpha) / beta;
    scale = 1.0 / (alpha - beta);
  }
  if (tid == 0) { tauv[k] = t; dvec[k] = x[0]; evec[k + 1] = beta; }
#pragma unroll
  for (int r = 0; r < RMAX; ++r) {
    const int i = k + tid + 1024 * r;
    if (i > k && i < n) {
      const double v = (i == k + 1) ? 1.0 : x[r] * scale;
      vnew[i] = v;
      if (i > k + 1) Wk[i] = v;
    }
  }
}

// Symmetric sweep over the UPPER triangle of the trailing block (rows/cols k+1..n-1; relative index ii = i-(k+1)):
//   x = W[i][j] - vprev[i] w[j] - w[i] vprev[j]   (pending update of reflector k-1; skipped when k == 0), j >= i,
// stored back, and the two halves of y = A22 v_k:
//   rowpart[c][i] = sum_{j in chunk c, j >= i} x_ij vnew[j]        colpart[g][j] = sum_{i in row group g, i < j} x_ij vnew[i]
// Grid: x = column chunk c (EIGH_CW columns), y = row group g (rg rows, a multiple of 32).  A CTA walks the 32-row blocks
// of its group that reach the chunk (warp w: rows 4w..4w+3 of the block, lanes along the contiguous j, 8 columns per
// lane), keeps its column sums in registers, and reduces them over its 8 warps at the end.  Half the bytes of a
// full-matrix sweep; every partial is written by exactly one CTA and summed later in a fixed order (deterministic).
__global__ void __launch_bounds__(256, 2)
eigh_pass_kernel(double* __restrict__ W, int n, int k, int rg, const double* __restrict__ vprev,
                 const double* __restrict__ wv, const double* __restrict__ vnew, double* __restrict__ rowpart,
                 double* __restrict__ colpart) {
  constexpr int QW = EIGH_CW / 32, ROWS = 4;
  __shared__ double s_col[8][EIGH_CW];
  eigh_pdl_sync();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool pending = k > 0;
  const int base = k + 1, nt = n - base;
  const int c = blockIdx.x, g = blockIdx.y;
  const int jj0 = c * EIGH_CW, jlast = min(jj0 + EIGH_CW, nt) - 1;     // relative column range of the chunk
  const int ii_begin = g * rg, ii_end = min(ii_begin + rg, nt);
  if (ii_begin > jlast) return;                                        // group entirely below the diagonal
  double vn[QW], vp[QW], wj[QW], colacc[QW];
#pragma unroll
  for (int q = 0; q < QW; ++q) {
    const int jj = jj0 + lane + 32 * q;
    const bool ok = jj < nt;
    vn[q] = ok ? vnew[base + jj] : 0.0;
    vp[q] = (ok && pending) ? vprev[base + jj] : 0.0;
    wj[q] = (ok && pending) ? wv[base + jj] : 0.0;
    colacc[q] = 0.0;
  }
  double* rp = rowpart + (long long)c * n + base;
  for (int rb = ii_begin; rb < ii_end && rb <= jlast; rb += 32) {
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
      const int ii = rb + ROWS * warp + r;
      if (ii >= ii_end || ii > jlast) continue;                       // warp-uniform
      double* row = W + (long long)(base + ii) * n + base + jj0 + lane;
      const double vni = vnew[base + ii];
      const double vi = pending ? vprev[base + ii] : 0.0, wi = pending ? wv[base + ii] : 0.0;
      double x[QW];
#pragma unroll
      for (int q = 0; q < QW; ++q) {
        const int jj = jj0 + lane + 32 * q;
        x[q] = (jj >= ii && jj < nt) ? row[32 * q] : 0.0;
      }
      double racc = 0.0;
#pragma unroll
      for (int q = 0; q < QW; ++q) {
        const int jj = jj0 + lane + 32 * q;
        if (jj >= ii && jj < nt) {
          if (pending) {
            x[q] = fma(-vi, wj[q], x[q]);
            x[q] = fma(-wi, vp[q], x[q]);
            row[32 * q] = x[q];
          }
          racc = fma(x[q], vn[q], racc);
          if (jj > ii) colacc[q] = fma(x[q], vni, colacc[q]);
        }
      }
      racc = warp_sum(racc);
      if (lane == 0) rp[ii] = racc;
    }
  }
#pragma unroll
  for (int q = 0; q < QW; ++q) s_col[warp][lane + 32 * q] = colacc[q];
  __syncthreads();
  {
    const int t = threadIdx.x, jj = jj0 + t;
    if (jj < nt) {
      double sacc = 0.0;
#pragma unroll
      for (int w2 = 0; w2 < 8; ++w2) sacc += s_col[w2][t];
      colpart[(long long)g * n + base + jj] = sacc;
    }
  }
}

// y[i] = sum of the sweep's partials in a fixed order: row parts of the chunks from the one holding the diagonal on,
// column parts of the row groups up to the one holding row i.
__global__ void __launch_bounds__(64)
eigh_ysum_kernel(const double* __restrict__ rowpart, const double* __restrict__ colpart, int n, int k, int rg,
                 double* __restrict__ y) {
  eigh_pdl_sync();
  const int base = k + 1, nt = n - base;
  const int ii = blockIdx.x * 64 + threadIdx.x;
  if (ii >= nt) return;
  const int nch = (nt + EIGH_CW - 1) / EIGH_CW;
  double acc = eigh_strided_sum(rowpart + base + ii, n, ii / EIGH_CW, nch, 0.0);
  acc = eigh_strided_sum(colpart + base + ii, n, 0, ii / rg + 1, acc);
  y[base + ii] = acc;
}

// (W + W^T)/2 in place (C~ is symmetric for a C4v state; rounding in the GEMMs that
// build it breaks that at the 1e-16 level; reading A15).
__global__ void symmetrize_inplace_kernel(double* __restrict__ W, int n) {
  const long long total = (long long)n * n;
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
       idx += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(idx / n), j = (int)(idx % n);
    if (j < i) {
      const double a = W[idx], b = W[(long long)j * n + i];
      const double s = 0.5 * (a + b);
      W[idx] = s; W[(long long)j * n + i] = s;
    }
  }
}

// eig[nc] ascending (the candidates: all n eigenvalues, or the k smallest followed by the k largest -- an
// eigenvalue of rank < k in |lambda| is always among those) -> lamsel[r] = the eigenvalue of rank r in decreasing |lambda| (ties: lower index
// first, i.e. numpy's stable argsort of -|lambda| on the ascending list), r < k.
// scal[0] = max_i (|d_i| + |e_i| + |e_{i+1}|), the norm bound used as pivot scale by the inverse iteration.
__global__ void eigh_select_kernel(const double* __restrict__ eig, int nc, int k, double* __restrict__ lamsel,
                                   const double* __restrict__ dvec, const double* __restrict__ evec, int n,
                                   double* __restrict__ scal) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < nc) {
    const double mine = fabs(eig[i]);
    int rank = 0;
    for (int j = 0; j < nc; ++j) {
      const double o = fabs(eig[j]);
      rank += (o > mine) || (o == mine && j < i);
    }
    if (rank < k) lamsel[rank] = eig[i];
  }
  if (blockIdx.x == 0) {
    __shared__ double sh[33];
    double mx = 0.0;
    for (int t = threadIdx.x; t < n; t += blockDim.x) {
      const double el = t > 0 ? fabs(evec[t]) : 0.0, er = t + 1 < n ? fabs(evec[t + 1]) : 0.0;
      mx = fmax(mx, fabs(dvec[t]) + el + er);
    }
    mx = block_max(mx, sh);
    if (threadIdx.x == 0) scal[0] = mx;
  }
}

__device__ __forceinline__ double eigh_rnd(unsigned i, unsigned c) {   // counter-based, in (-1, 1)
  unsigned long long z = ((unsigned long long)i << 32 | c) + 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  z ^= z >> 31;
  return ((double)(z >> 11) + 0.5) * (2.0 / 9007199254740992.0) - 1.0;
}

// Inverse iteration for column c: (T - lam_c) x = rhs, `iters` times from a random start, x normalised
// after every solve.  T - lam = P L U by Gaussian elimination with partial pivoting (two
// superdiagonals in U); the elimination is replayed on the right-hand side in the same sweep.
// Z, U0, U1, U2: n x k row-major (threads of a warp touch consecutive addresses).
__global__ void eigh_invit_kernel(const double* __restrict__ dvec, const double* __restrict__ evec, int n,
                                  const double* __restrict__ lamsel, int k, const double* __restrict__ scal,
                                  double* __restrict__ Z, double* __restrict__ U0, double* __restrict__ U1,
                                  double* __restrict__ U2, int iters) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= k) return;
  const double lam = lamsel[c];
  const double tiny = fmax(2.220446049250313e-16 * scal[0], 1e-300);
  // rhs of sweep `it` = sc * (x of sweep it-1); sweep 0: random numbers generated on the fly
  double sc = 1.0;
  for (int it = 0; it < iters; ++it) {
    double p0 = dvec[0] - lam, p1 = n > 1 ? evec[1] : 0.0, p2 = 0.0;
    double r = it ? sc * Z[c] : eigh_rnd(0u, (unsigned)c);
    for (int i = 0; i + 1 < n; ++i) {
      const double cc = evec[i + 1], a = dvec[i + 1] - lam, b = i + 2 < n ? evec[i + 2] : 0.0;
      const double yn = it ? sc * Z[(long long)(i + 1) * k + c] : eigh_rnd((unsigned)(i + 1), (unsigned)c);
      double u0, u1, u2, ri, n0, n1, nr;
      if (fabs(p0) >= fabs(cc)) {
        if (fabs(p0) < tiny) p0 = p0 < 0.0 ? -tiny : tiny;
        const double mlt = cc / p0;
        u0 = p0; u1 = p1; u2 = p2; ri = r;
        n0 = fma(-mlt, p1, a); n1 = fma(-mlt, p2, b); nr = fma(-mlt, r, yn);
      } else {
        const double mlt = p0 / cc;
        u0 = cc; u1 = a; u2 = b; ri = yn;
        n0 = fma(-mlt, a, p1); n1 = fma(-mlt, b, p2); nr = fma(-mlt, yn, r);
      }
      const long long o = (long long)i * k + c;
      if (it == 0) { U0[o] = 1.0 / u0; U1[o] = u1; U2[o] = u2; }      // the factors do not depend on the rhs
      Z[o] = ri;
      p0 = n0; p1 = n1; p2 = 0.0; r = nr;
    }
    if (fabs(p0) < tiny) p0 = p0 < 0.0 ? -tiny : tiny;
    {
      const long long o = (long long)(n - 1) * k + c;
      if (it == 0) { U0[o] = 1.0 / p0; U1[o] = 0.0; U2[o] = 0.0; }
      Z[o] = r;
    }
    // back substitution; the growth is bounded by 1 / (eps ||T||) per sweep, so the sum of squares cannot overflow
    double x1 = 0.0, x2 = 0.0, ss = 0.0;
    for (int i = n - 1; i >= 0; --i) {
      const long long o = (long long)i * k + c;
      double x = Z[o];
      x = fma(-U1[o], x1, x);
      x = fma(-U2[o], x2, x);
      x *= U0[o];
      Z[o] = x;
      x2 = x1; x1 = x;
      ss = fma(x, x, ss);
    }
    sc = ss > 0.0 ? 1.0 / sqrt(ss) : 1.0;
  }
  for (int i = 0; i < n; ++i) Z[(long long)i * k + c] *= sc;
}

// U = H_0 H_1 ... H_{n-3} U, reflector k = I - tau_k v v^T with v[k+1] = 1, v[j] = W[k][j] (j > k+1).
// CTA b owns columns 2b, 2b+1 of U (n x ldu) in shared memory; thread t owns rows t, t + 1024, ...
// for the whole kernel, so only the two dot products need a block-wide exchange per reflector; the
// next reflector row is prefetched into L1 while the current one is applied.
__global__ void __launch_bounds__(1024, 1)
eigh_backtransform_kernel(const double* __restrict__ W, const double* __restrict__ tauv, int n,
                          double* __restrict__ U, int ldu, int ncols) {
  extern __shared__ __align__(16) double bsm[];      // x0[n], x1[n]
  __shared__ double part[2][2][32];
  double* x0 = bsm;
  double* x1 = bsm + n;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c0 = 2 * blockIdx.x, c1 = c0 + 1;
  const bool two = c1 < ncols;
  for (int i = tid; i < n; i += 1024) {
    x0[i] = U[(long long)i * ldu + c0];
    x1[i] = two ? U[(long long)i * ldu + c1] : 0.0;
  }
  int buf = 0;
  for (int k = n - 3; k >= 0; --k) {
    const double* Wk = W + (long long)k * n;
    if (k > 0) {                                     // next reflector row into L1, one request per 128-byte line
      const double* Wn = Wk - n;
      for (int i = (k & ~15) + 16 * tid; i < n + 15; i += 16 * 1024)
        asm volatile("prefetch.global.L1 [%0];" ::"l"(Wn + min(i, n - 1)));
    }
    const double tau = tauv[k];
    if (tau == 0.0) continue;
    const int ifirst = tid > k ? tid : tid + ((k - tid) / 1024 + 1) * 1024;     // first owned row > k
    double a0 = 0.0, a1 = 0.0;
    for (int i = ifirst; i < n; i += 1024) {
      const double v = (i == k + 1) ? 1.0 : Wk[i];
      a0 = fma(v, x0[i], a0);
      a1 = fma(v, x1[i], a1);
    }
    a0 = warp_sum(a0); a1 = warp_sum(a1);
    if (lane == 0) { part[buf][0][warp] = a0; part[buf][1][warp] = a1; }
    __syncthreads();
    double s0 = part[buf][0][lane], s1 = part[buf][1][lane];
    s0 = warp_sum(s0) * tau; s1 = warp_sum(s1) * tau;
    for (int i = ifirst; i < n; i += 1024) {
      const double v = (i == k + 1) ? 1.0 : Wk[i];
      x0[i] = fma(-s0, v, x0[i]);
      x1[i] = fma(-s1, v, x1[i]);
    }
    buf ^= 1;
  }
  for (int i = tid; i < n; i += 1024) {
    U[(long long)i * ldu + c0] = x0[i];
    if (two) U[(long long)i * ldu + c1] = x1[i];
  }
}

// One CTA per column: the component of largest magnitude (first one on ties, numpy's argmax) is made positive.
__global__ void __launch_bounds__(256)
eigh_sign_kernel(double* __restrict__ U, int n, int ldu) {
  __shared__ double sv[256];
  __shared__ int si[256];
  const int c = blockIdx.x, tid = threadIdx.x;
  double best = -1.0; int bi = 0x7fffffff;
  for (int i = tid; i < n; i += 256) {
    const double a = fabs(U[(long long)i * ldu + c]);
    if (a > best) { best = a; bi = i; }
  }
  sv[tid] = best; si[tid] = bi;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (tid < s) {
      const double o = sv[tid + s]; const int oi = si[tid + s];
      if (o > sv[tid] || (o == sv[tid] && oi < si[tid])) { sv[tid] = o; si[tid] = oi; }
    }
    __syncthreads();
  }
  const bool flip = U[(long long)si[0] * ldu + c] < 0.0;
  __syncthreads();
  if (flip)
    for (int i = tid; i < n; i += 256) U[(long long)i * ldu + c] = -U[(long long)i * ldu + c];
}

// out (k x k) = diag(lam)
__global__ void diag_matrix_kernel(const double* __restrict__ lam, int k, double* __restrict__ out) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < k * k) out[idx] = (idx / k == idx % k) ? lam[idx / k] : 0.0;
}

// fn.[48] PAPER.md:132: boundary from the bulk tensor, open bra/ket legs contracted:
//   C0[(d d'),(r r')]        = sum_{s,u,l} A[s,u,l,d,r] A[s,u,l,d',r']
//   T0[(l l'),(d d'),(r r')] = sum_{s,u}   A[s,u,l,d,r] A[s,u,l',d',r']
// One thread per output element (b^2 + b^3 elements, d D^2 resp. d D terms each).
__global__ void bulk_init_kernel(const double* __restrict__ A, int d, int D, double* __restrict__ C0,
                                 double* __restrict__ T0) {
  const int b = D * D;
  const long long nC = (long long)b * b, nT = nC * b;
  const long long s1 = (long long)D * D * D * D;      // stride of s
  const long long su = (long long)D * D * D, sl = (long long)D * D;
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < nC + nT;
       idx += (long long)gridDim.x * blockDim.x) {
    if (idx < nC) {
      const int dd = (int)(idx / b), rr = (int)(idx % b);
      const int dk = dd / D, db = dd % D, rk = rr / D, rb = rr % D;
      double acc = 0.0;
      for (int s = 0; s < d; ++s)
        for (int u = 0; u < D; ++u)
          for (int l = 0; l < D; ++l) {
            const double* base = A + s * s1 + u * su + l * sl;
            acc = fma(base[dk * D + rk], base[db * D + rb], acc);
          }
      C0[idx] = acc;
    } else {
      const long long t = idx - nC;
      const int ll = (int)(t / nC), dd = (int)((t / b) % b), rr = (int)(t % b);
      const int lk = ll / D, lb = ll % D, dk = dd / D, db = dd % D, rk = rr / D, rb = rr % D;
      double acc = 0.0;
      for (int s = 0; s < d; ++s)
        for (int u = 0; u < D; ++u) {
          const double* base = A + s * s1 + u * su;
          acc = fma(base[lk * sl + dk * D + rk], base[lb * sl + db * D + rb], acc);
        }
      T0[t] = acc;
    }
  }
}

}  // namespace qk
