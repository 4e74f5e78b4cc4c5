// K8: corner spectrum.  s = descending |eigenvalues| of the symmetric, Frobenius-
// normalised corner C (reading A6), delta = max_i |s_i - s_prev_i|.
//
// Algorithm (one CTA, chi <= a few hundred): Householder tridiagonalisation of a
// working copy W (lower triangle referenced, kept in global/L2), then every
// eigenvalue by Sturm-sequence bisection (one thread per eigenvalue), then a
// rank sort.  Bisection gives each eigenvalue to ~2 ulp of ||C|| = 1, which is
// what the convergence test (tol 1e-10..1e-12 absolute) needs.
#pragma once
#include <stdint.h>
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

// ------------------------------------------------------------------------------
// Round-2 tridiagonalisation (n <= TRI2_MAX_N): same storage (packed lower triangle in shared memory), organised
// around what bounds this kernel -- one SM, n dependent Householder steps, so instruction count and barriers per
// step, not bandwidth (ncu on the round-1 kernel and on a first warp-per-row rewrite: issue slots busy, 12 % of the
// instructions FP64; profiles/r2_k8_spectrum.md):
//   * ONE THREAD PER COLUMN j.  p_j = sum_i A_sym[i][j] u_i is a private loop (no warp reduction per row); the element
//     (i, j) is read at tri(i) + j for i >= j (consecutive threads, consecutive addresses) and at tri(j) + i for
//     i < j -- triangular numbers are a complete residue system modulo 16, so the 16 threads of a half-warp hit 16
//     different 8-byte banks there too: conflict-free in both directions without a second copy of the matrix;
//   * u is never copied: it is column k of the matrix itself (read as a broadcast), its head u_{k+1} = alpha - beta
//     is a register.  The reflector is un-normalised, H = I - gamma u u^T, gamma = 1 / (beta (beta - alpha)): one
//     rsqrt and one reciprocal per step, computed redundantly by every warp (no broadcast barrier);
//   * the rank-2 update A -= u w^T + w u^T runs down the thread's own column with w_i = p_i - (gamma/2)(p.u) u_i
//     formed on the fly.
// Two barriers per step.  Output as tridiag_smem_kernel (d, e; e[0] = 0); the similarity transform differs from
// LAPACK's only in the scaling of u, so the eigenvalues agree to rounding.
constexpr int TRI2_NT = 1024, TRI2_MAX_N = 216, TRI2_MAXSUB = 8, TRI2_MAXCG = (TRI2_MAX_N + 31) / 32;
__host__ __device__ inline size_t tri2_smem_bytes(int n) {
  return sizeof(double) * ((size_t)n * (n + 1) / 2 + 1 + (4 + TRI2_MAXSUB) * (size_t)n + 16);
}

// 1024 threads = 32 warps, four barriers per step.  What bounds this kernel is the ISSUE rate of one SM (ncu: the
// matrix-vector and update loops are "not selected" / issue limited once all 32 warps work), so scalar work is done
// by ONE warp and broadcast through shared memory (a barrier costs ~70 cycles, redundant scalar code in 32 warps
// ~1000), and the two O(n^2) loops are written for few instructions per element (contiguous row chunks per warp,
// immediate offsets, incremental triangular offsets):
//   R  warp 0: reflector scalars of column k (one rsqrt, one reciprocal), u_{k+1} written in place, and the table
//      that deals the warps out for phase U                                                              -- barrier
//   M  p = A u: the active column groups (32 columns each) share the warps evenly, the wpg <= 8 warps of a group
//      take contiguous row chunks and leave partial sums part[sub][j]                                    -- barrier
//   C  thread j sums the partials in a fixed order: p_j = gamma sum_sub part[sub][j]; p.u                -- barrier
//   U  rank-2 update of the lower triangle, warps dealt out to the column groups in proportion to the groups'
//      heights (the first group's columns are n - k rows tall, the last one's a few); the owner of column k+1 also
//      leaves it as the next u                                                                           -- barrier
__device__ __forceinline__ void
tridiag_smem2_body(double* tsm, const double* Cmat, int n, double* dvec, double* evec,
                   long long* prof /* null, or 8 cycle counters of the phases (thread 0) */) {
  double2* up0 = reinterpret_cast<double2*>(tsm);               // 2 x n pairs (u_i, p_i), double-buffered over the steps
  double* part = tsm + 4 * n;                                   // TRI2_MAXSUB x n partial sums of A u
  double* red = part + TRI2_MAXSUB * n;                         // 8: per-warp partial sums of p.u
  double* sc = red + 8;                                         // [0] gamma (0: nothing to eliminate)
  double* L = red + 16;                                         // n(n+1)/2
  __shared__ int tab[2][32];                                    // warp table of phase U, rebuilt every 8 steps (two copies)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  long long tp[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tc = 0;
#define TRI_TICK(i) do { if (prof && tid == 0) { const long long t_ = clock64(); tp[i] += t_ - tc; tc = t_; } } while (0)
  if (prof && tid == 0) tc = clock64();
  for (int i = warp; i < n; i += TRI2_NT / 32)
    for (int j = lane; j <= i; j += 32) {
      const double v = Cmat[(long long)i * n + j];
      L[tri_off(i) + j] = v;
      if (j == 0) up0[i].x = v;
    }
  __syncthreads();
  TRI_TICK(0);
  const int ncgt = (n + 31) >> 5;
  // ---- R (warp 0): reflector of column k (rows k+1 .. n-1) from the column left in up0 + (k & 1) n, and every 8 steps
  // the warp table of phase U.  Runs one step AHEAD: R(k+1) beside the rank-2 update of step k (U2 below), so the scalar
  // chain (norm -> rsqrt -> reciprocal, ~1 us) is off the critical path.
  auto reflector = [&](int k) {
    double2* up = up0 + (k & 1) * n;
    const int c0 = (k + 1) >> 5, ncg = ncgt - c0;
    double acc = 0.0;
    for (int i = k + 2 + lane; i < n; i += 32) { const double x = up[i].x; acc = fma(x, x, acc); }
    const double tail2 = warp_sum(acc);
    const double alpha = up[k + 1].x;
    __syncwarp();
    // nothing to eliminate: H = I.  Entries below 1e-140 in magnitude are dropped rather than eliminated: gamma ~
    // 1 / tail2 would overflow, and the perturbation is 120 orders below rounding for ||C|| ~ 1
    if (!(tail2 > 1e-280)) {
      if (lane == 0) { dvec[k] = L[tri_off(k) + k]; evec[k + 1] = alpha; sc[0] = 0.0; }
    } else {
      const double s2 = fma(alpha, alpha, tail2);
      const double sigma = s2 * rsqrt(s2);                     // 1-2 ulp: only perturbs e_{k+1} at rounding level
      const double beta = alpha >= 0.0 ? -sigma : sigma;
      const double gamma = __drcp_rn(fma(-alpha, beta, s2));   // 1 / (beta (beta - alpha)),  beta^2 = s2
      if (lane == 0) {
        dvec[k] = L[tri_off(k) + k]; evec[k + 1] = beta; sc[0] = gamma;
        up[k + 1].x = alpha - beta;                            // u_{k+1}: H = I - gamma u u^T, u = x - beta e_1
      }
    }
    // every 8 steps: deal warps 1..31 out to the active column groups for phase U2, in proportion to the groups'
    // heights h_c = n - max(32 c, k+1) (a table that is up to 7 steps old only balances slightly worse: rows and
    // columns that have left the active block are skipped by the lanes themselves)
    if ((k & 7) == 0) {
      const int c = c0 + lane;                                  // lane <-> active column group
      const int h = (lane < ncg) ? n - ((c << 5) > k + 1 ? (c << 5) : k + 1) : 0;
      int cum = h;
#pragma unroll
      for (int o = 1; o < 8; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, cum, o); if (lane >= o) cum += v; }
      const int H = __shfl_sync(0xffffffffu, cum, ncg - 1);
      int B = (lane == ncg - 1) ? 31 : (int)((float)cum * __fdividef(31.0f, (float)H));
      int m = B - lane;                                         // at least one warp per group: B_c >= B_c' + (c - c')
#pragma unroll
      for (int o = 1; o < 8; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, m, o); if (lane >= o) m = m > v ? m : v; }
      B = m + lane;
      const int room = 31 - (ncg - 1 - lane);                   // ... and one left for every later group
      B = B < room ? B : room;
      int t = 0xff;
      for (int cc = 0; cc < ncg; ++cc) {
        const int hi = __shfl_sync(0xffffffffu, B, cc), lo = cc ? __shfl_sync(0xffffffffu, B, cc - 1) : 0;
        const int hh = __shfl_sync(0xffffffffu, h, cc);
        if (lane >= lo && lane < hi) {
          const int cnt = hi - lo;
          t = (c0 + cc) | ((lane - lo) << 8) | (((hh + cnt - 1) / cnt) << 16);        // group, sub, rows per warp
        }
      }
      tab[(k >> 3) & 1][lane] = t;                              // slot s <-> warp s + 1
    }
  };
  if (n > 2) {
    if (warp == 0) reflector(0);
    __syncthreads();
  }
  TRI_TICK(1);
  for (int k = 0; k < n - 2; ++k) {
    double2* up = up0 + (k & 1) * n;
    double2* upn = up0 + ((k + 1) & 1) * n;
    const int c0 = (k + 1) >> 5, ncg = ncgt - c0;
    const bool more = k + 1 < n - 2;                             // there is a next step
    const double gamma = sc[0];
    if (gamma == 0.0) {
      for (int i = k + 2 + tid; i < n; i += TRI2_NT) upn[i].x = L[tri_off(i) + k + 1];
      __syncthreads();
      if (more && warp == 0) reflector(k + 1);
      __syncthreads();
      continue;
    }
    // ---- M: partial sums of A u
    const int wpg = ncg <= 4 ? 8 : (ncg == 5 ? 6 : (ncg == 6 ? 5 : 4));
    {
      const int g = wpg == 8 ? warp >> 3 : (wpg == 6 ? warp / 6 : (wpg == 5 ? warp / 5 : warp >> 2));
      const int sub = warp - g * wpg;
      if (g < ncg) {
        const int jlo = (c0 + g) << 5, jhi = jlo + 32 < n ? jlo + 32 : n;
        const int j = jlo + lane;
        const int jc = j < k + 1 ? k + 1 : (j < n ? j : n - 1);  // out-of-range lanes compute a valid column (discarded)
        const double* Lrow = L + tri_off(jc);                    // element (jc, i), i <= jc
        const double* Lcol = L + jc;                             // element (i, jc) at Lcol[tri(i)], i >= jc
        const int na = n - (k + 1);
        const int chunk = wpg == 8 ? (na + 7) >> 3 : (wpg == 6 ? (na + 5) / 6 : (wpg == 5 ? (na + 4) / 5 : (na + 3) >> 2));
        const int r0 = k + 1 + sub * chunk, r1 = r0 + chunk < n ? r0 + chunk : n;
        double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
        int i = r0;
        {                                                        // rows above the group's columns: my row, contiguous
          const int e = r1 < jlo ? r1 : jlo;
          for (; i + 4 <= e; i += 4) {
            a0 = fma(Lrow[i], up[i].x, a0);
            a1 = fma(Lrow[i + 1], up[i + 1].x, a1);
            a2 = fma(Lrow[i + 2], up[i + 2].x, a2);
            a3 = fma(Lrow[i + 3], up[i + 3].x, a3);
          }
          for (; i < e; ++i) a0 = fma(Lrow[i], up[i].x, a0);
        }
        {                                                        // rows inside the group's columns: row or column
          const int e = r1 < jhi ? r1 : jhi;
          int off = tri_off(i);
          for (; i + 2 <= e; i += 2) {
            a1 = fma(i >= jc ? Lcol[off] : Lrow[i], up[i].x, a1);
            a2 = fma(i + 1 >= jc ? Lcol[off + i + 1] : Lrow[i + 1], up[i + 1].x, a2);
            off += 2 * i + 3;
          }
          if (i < e) { a3 = fma(i >= jc ? Lcol[off] : Lrow[i], up[i].x, a3); ++i; }
        }
        if (i < r1) {                                            // rows below: my column, incremental offsets
          int off = tri_off(i);
          for (; i + 4 <= r1; i += 4) {
            const int o1 = off + i + 1, o2 = o1 + i + 2, o3 = o2 + i + 3;
            a0 = fma(Lcol[off], up[i].x, a0);
            a1 = fma(Lcol[o1], up[i + 1].x, a1);
            a2 = fma(Lcol[o2], up[i + 2].x, a2);
            a3 = fma(Lcol[o3], up[i + 3].x, a3);
            off = o3 + i + 4;
          }
          for (; i < r1; ++i) { a0 = fma(Lcol[off], up[i].x, a0); off += i + 1; }
        }
        if (j >= k + 1 && j < n) part[sub * n + j] = (a0 + a1) + (a2 + a3);
      }
    }
    TRI_TICK(2);
    __syncthreads();
    // ---- C: p_j, p.u
    if (warp < 8) {
      double pj = 0.0, uj = 0.0;
      if (tid < n && tid > k) {
        double sum = 0.0;
        for (int q = 0; q < wpg; ++q) sum += part[q * n + tid];
        pj = gamma * sum;
        uj = up[tid].x;
        up[tid].y = pj;
      }
      const double q = warp_sum(pj * uj);
      if (lane == 0) red[warp] = q;
    }
    TRI_TICK(3);
    __syncthreads();
    // ---- U: A -= u w^T + w u^T: x = A_ij - u_i (p_j - 2 cf u_j) - p_i u_j,  cf = (gamma/2) p.u
    double pu = 0.0;
#pragma unroll
    for (int w = 0; w < 8; ++w) pu += red[w];
    const double cf = 0.5 * gamma * pu;
    // U1: column k+1 first (one element per thread): it is the next step's u
    {
      const int i = k + 1 + tid;
      if (i < n) {
        const double2 mine = up[k + 1], ui = up[i];
        const double aj = fma(-2.0 * cf, mine.x, mine.y), bj = mine.x;
        double* e = L + tri_off(i) + k + 1;
        const double x = fma(-ui.y, bj, fma(-ui.x, aj, *e));
        *e = x;
        upn[i].x = x;
      }
    }
    __syncthreads();
    TRI_TICK(4);
    // U2 (warps 1..31): the columns right of k+1;  R (warp 0): the reflector of the next step
    if (warp == 0) {
      if (more) reflector(k + 1);
    } else {
      const int t = tab[(k >> 3) & 1][warp - 1];
      const int cgm = t & 0xff;
      if (cgm != 0xff) {
        const int sub = (t >> 8) & 0xff, chunk = t >> 16;
        const int jlo = cgm << 5;
        const int j = jlo + lane;
        const bool active = j > k + 1 && j < n;
        const int k8 = (k & ~7) + 1;                             // the table was built at step k & ~7
        const int start = jlo > k8 ? jlo : k8;
        const int r0 = start + sub * chunk, r1 = r0 + chunk < n ? r0 + chunk : n;
        if (active) {
          const double2 mine = up[j];
          const double aj = fma(-2.0 * cf, mine.x, mine.y), bj = mine.x;
          double* Lc = L + j;
          int i = r0 > j ? r0 : j;                               // rows above my diagonal element are not mine
          if (i < r1) {
            int off = tri_off(i);
            for (; i + 4 <= r1; i += 4) {
              const int o1 = off + i + 1, o2 = o1 + i + 2, o3 = o2 + i + 3;
              const double2 u0 = up[i], u1v = up[i + 1], u2 = up[i + 2], u3 = up[i + 3];
              const double x0 = fma(-u0.y, bj, fma(-u0.x, aj, Lc[off]));
              const double x1 = fma(-u1v.y, bj, fma(-u1v.x, aj, Lc[o1]));
              const double x2 = fma(-u2.y, bj, fma(-u2.x, aj, Lc[o2]));
              const double x3 = fma(-u3.y, bj, fma(-u3.x, aj, Lc[o3]));
              Lc[off] = x0; Lc[o1] = x1; Lc[o2] = x2; Lc[o3] = x3;
              off = o3 + i + 4;
            }
            for (; i < r1; ++i) {
              const double2 ui = up[i];
              const double x = fma(-ui.y, bj, fma(-ui.x, aj, Lc[off]));
              Lc[off] = x;
              off += i + 1;
            }
          }
        }
      }
    }
    TRI_TICK(4);
    __syncthreads();
    TRI_TICK(5);
  }
  if (tid == 0) {
    if (n >= 2) {
      dvec[n - 2] = L[tri_off(n - 2) + n - 2];
      evec[n - 1] = L[tri_off(n - 1) + n - 2];
    }
    dvec[n - 1] = L[tri_off(n - 1) + n - 1];
    evec[0] = 0.0;
    if (prof) for (int i = 0; i < 8; ++i) prof[i] = tp[i];
  }
#undef TRI_TICK
}

__global__ void __launch_bounds__(TRI2_NT, 1)
tridiag_smem2_kernel(const double* __restrict__ Cmat, int n, double* __restrict__ dvec, double* __restrict__ evec,
                     long long* __restrict__ prof) {
  extern __shared__ __align__(16) double tsm[];
  tridiag_smem2_body(tsm, Cmat, n, dvec, evec, prof);
}

// Sturm count without divisions: number of eigenvalues < x of the tridiagonal whose SCALED entries (all magnitudes
// <= ~2) are de[i] = (d_i, e_i^2), from the sign changes of the leading principal minors
//   p_i = (d_i - x) p_{i-1} - e_i^2 p_{i-2}
// (q_i = p_i / p_{i-1} is the pivot sequence of sturm_count above: q_i < 0 <=> p_i and p_{i-1} differ in sign).  The
// dependent chain is one FMA per row instead of one FP64 division (~15x shorter).  Every computed p_i is the exact
// minor of a matrix with relatively perturbed entries (backward stable); only signs are used, so p is renormalised by
// an exact power of two every 4 rows (magnitudes then stay within 2^+-600 of 1).  d_i - x == 0 is replaced by 2^-100
// (a perturbation of x far below rounding at this scaling); an exact zero minor counts as a sign change.
// LEAN = true (the 1024-thread kernels, 64 registers per thread): groups of four rows without the look-ahead fetch -- the
// eight-row version's 64 staging registers would spill there.
template <bool LEAN = false>
__device__ __forceinline__ int sturm_count_minors(const double2* __restrict__ de, int n, double x) {
  // Few instructions per row (the count is issue-bound as soon as two warps share a scheduler): the sign changes are
  // counted on the sign words (an exact zero counts as positive: the row after it has the sign opposite to the row
  // before it, so a zero adds one change whichever sign it is given); d_i - x = 0 is moved to 2^-100 by an addition
  // instead of a compare-and-select, so that a decoupled row (e = 0) cannot zero the sequence.
  double p0 = 1.0;
  double p1 = (de[0].x - x) + 0x1p-100;
  int sprev = __double2hiint(p1);
  int cnt = (int)((unsigned)sprev >> 31);
  int i = 1;
  // rows in groups of eight: the group's (d_i - x, -e_i^2) are formed ahead of the dependent chain (one FMA per row),
  // and the next group's rows are fetched from shared memory before the chain of the current one starts
  if (LEAN) {
    for (; i + 4 <= n; i += 4) {
      double2 v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) v[u] = de[i + u];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const double tt = (v[u].x - x) + 0x1p-100;
        const double pn = fma(tt, p1, -v[u].y * p0);
        const int sn = __double2hiint(pn);
        cnt += (int)((unsigned)(sn ^ sprev) >> 31);
        sprev = sn; p0 = p1; p1 = pn;
      }
      const int e0 = __double2hiint(p0) & 0x7ff00000, e1 = __double2hiint(p1) & 0x7ff00000;
      const int em = e0 > e1 ? e0 : e1;
      if ((unsigned)(em - ((1023 - 64) << 20)) > (unsigned)(128 << 20)) {
        if (em == 0) { p0 = 0.0; p1 = sprev < 0 ? -1.0 : 1.0; }
        else {
          const int e = (em >> 20) - 1023;
          const int ee = e > 1000 ? 1000 : (e < -1000 ? -1000 : e);
          const double sc = __hiloint2double((1023 - ee) << 20, 0);
          p0 *= sc; p1 *= sc;
        }
      }
    }
  }
  double2 w[8];
  if (!LEAN && i + 8 <= n) {
#pragma unroll
    for (int u = 0; u < 8; ++u) w[u] = de[i + u];
  }
  for (; !LEAN && i + 8 <= n; i += 8) {
    double tt[8], ne[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) { tt[u] = (w[u].x - x) + 0x1p-100; ne[u] = -w[u].y; }
    if (i + 16 <= n) {
#pragma unroll
      for (int u = 0; u < 8; ++u) w[u] = de[i + 8 + u];
    }
    asm volatile("" ::: "memory");               // keeps the loads above ahead of the chain below
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const double pn = fma(tt[u], p1, ne[u] * p0);
      const int sn = __double2hiint(pn);
      cnt += (int)((unsigned)(sn ^ sprev) >> 31);
      sprev = sn; p0 = p1; p1 = pn;
    }
    // renormalise by 2^-e, e = the larger exponent of p0, p1 (growth per row <= 3, shrinkage per row can be ~1e-17
    // in a block of tiny rows: eight rows stay far from overflow and underflow); integer test on the exponent fields
    const int e0 = __double2hiint(p0) & 0x7ff00000, e1 = __double2hiint(p1) & 0x7ff00000;
    const int em = e0 > e1 ? e0 : e1;
    if ((unsigned)(em - ((1023 - 64) << 20)) > (unsigned)(128 << 20)) {
      if (em == 0) { p0 = 0.0; p1 = sprev < 0 ? -1.0 : 1.0; }           // both zero (or denormal): decoupled block, restart
      else {
        const int e = (em >> 20) - 1023;
        const int ee = e > 1000 ? 1000 : (e < -1000 ? -1000 : e);
        const double sc = __hiloint2double((1023 - ee) << 20, 0);
        p0 *= sc; p1 *= sc;
      }
    }
  }
  for (; i < n; ++i) {
    const double2 v = de[i];
    const double tt = (v.x - x) + 0x1p-100;
    const double pn = fma(tt, p1, -v.y * p0);
    const int sn = __double2hiint(pn);
    cnt += (int)((unsigned)(sn ^ sprev) >> 31);
    sprev = sn; p0 = p1; p1 = pn;
  }
  return cnt;
}

// Eigenvalues of the tridiagonal by warp-multisection: warp w of block B finds
// eigenvalue number idx = 8 B + w (ascending; see `ke` for the partial mode).  Each iteration the 32 lanes evaluate
// the Sturm count at 32 interior points of [a, b], shrinking the bracket 33-fold
// (about 11 iterations to the last ulp instead of ~55 bisection steps).
// Block-wide set-up of the multisection: de[i] = (d_i, e_i^2) of the problem scaled by an exact power of two so that every
// entry has magnitude <= 1 (the minors recurrence of sturm_count_minors then grows by at most ~2.5 per row), the
// Gershgorin interval [glo, ghi] of the scaled problem, and the factor isc that scales eigenvalues back.
__device__ __forceinline__ void multisect_setup(const double* dvec, const double* evec, int n, double2* de, double* red,
                                                double& glo, double& ghi, double& isc) {
  const int tid = threadIdx.x;
  double lo = INFINITY, hi = -INFINITY;
  for (int i = tid; i < n; i += blockDim.x) {                  // Gershgorin bounds
    const double el = i > 0 ? fabs(evec[i]) : 0.0, er = i + 1 < n ? fabs(evec[i + 1]) : 0.0, di = dvec[i];
    lo = fmin(lo, di - el - er);
    hi = fmax(hi, di + el + er);
  }
  ghi = block_max(hi, red);
  glo = -block_max(-lo, red);
  const double bnd = fmax(fabs(glo), fabs(ghi));
  int ex = 0;
  if (bnd > 0.0 && bnd < INFINITY) { frexp(bnd, &ex); }
  ex = ex > 1000 ? 1000 : (ex < -1000 ? -1000 : ex);
  const double sc = ldexp(1.0, -ex);
  isc = ldexp(1.0, ex);
  for (int i = tid; i < n; i += blockDim.x) {
    const double e = i > 0 ? evec[i] * sc : 0.0;
    de[i] = make_double2(dvec[i] * sc, e * e);
  }
  __syncthreads();
  glo *= sc; ghi *= sc;
  const double bs = fmax(fabs(glo), fabs(ghi));
  glo -= 2.0 * 2.220446049250313e-16 * bs * n + 0x1p-90;
  ghi += 2.0 * 2.220446049250313e-16 * bs * n + 0x1p-90;
}

// One warp: eigenvalue number idx (ascending) of the scaled problem by 33-way multisection.
// Stops when the bracket is narrower than 2^-54 of the spectrum's bound (the scaled problem has |lambda| <= 1): the
// tridiagonalisation's own backward error is n eps ||C||, so resolving the tiny eigenvalues to full RELATIVE accuracy
// (up to twice as many rounds) buys nothing for s, delta or the inverse-iteration shifts.
template <bool LEAN = false>
__device__ __forceinline__ double multisect_warp(const double2* de, int n, int idx, double glo, double ghi) {
  const int lane = threadIdx.x & 31;
  double a = glo, b = ghi;
  for (int it = 0; it < 64; ++it) {
    if (b - a <= 0x1p-54) break;
    const double h = (b - a) * (1.0 / 33.0);                    // (any interior points do: no division in the round)
    const double x = a + (lane + 1) * h;
    const bool inside = x > a && x < b;
    int cnt = inside ? sturm_count_minors<LEAN>(de, n, x) : (x >= b ? n : 0);
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
  return 0.5 * (a + b);
}

__global__ void __launch_bounds__(256)
multisect_kernel(const double* __restrict__ dvec, const double* __restrict__ evec, int n,
                 double* __restrict__ eig_out, int ke = 0) {
  extern __shared__ __align__(16) double msm[];               // de[n] = (d_i, e_i^2) scaled, red[33]
  double2* de = reinterpret_cast<double2*>(msm); double* red = msm + 2 * n;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double glo, ghi, isc;
  multisect_setup(dvec, evec, n, de, red, glo, ghi, isc);
  // ke > 0 (and 2 ke < n): only the ke smallest and the ke largest eigenvalues, written compactly
  // (slot c < ke: eigenvalue c; slot c >= ke: eigenvalue n - 2 ke + c) -- the eigen step's candidates.
  const int slot = blockIdx.x * (blockDim.x >> 5) + warp;
  const bool part = ke > 0 && 2 * ke < n;
  if (slot >= (part ? 2 * ke : n)) return;
  const int idx = (part && slot >= ke) ? n - 2 * ke + slot : slot;
  const double lam = multisect_warp(de, n, idx, glo, ghi);
  if (lane == 0) eig_out[slot] = lam * isc;
}

// One block, blockDim.x >= n: s = sorted |eig| (descending), delta vs s_prev.
// blockDim.x >= n.  lam[n] (shared): the eigenvalues; s = sorted |lam| (descending), delta vs s_prev.
// host_delta / host_flag (may be null): mapped pinned host words that receive delta and the NaN / zero-norm flag of K7
// (dev_flag) straight from the kernel, so that the overlapped run driver needs no copies after K8.
__device__ __forceinline__ void spectrum_finalize_body(const double* lam, double* red, int n, double* s_out,
                                                       double* s_prev, double* delta_out, int update_prev,
                                                       double* hist, const int* hist_n, double* host_delta = nullptr,
                                                       int* host_flag = nullptr, const int* dev_flag = nullptr) {
  const int tid = threadIdx.x;
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
  if (tid == 0) {
    delta_out[0] = dmax;
    if (host_delta) { host_delta[0] = dmax; host_flag[0] = dev_flag[0]; }
    if (hist && update_prev && *hist_n > 0) hist[(size_t)((*hist_n - 1) % 4096) * 4] = dmax;   // this step's record
  }
  __syncthreads();
  if (update_prev && tid < n) s_prev[tid] = s_out[tid];
}

// One block, blockDim.x >= n: s = sorted |eig| (descending), delta vs s_prev.
__global__ void spectrum_finalize_kernel(const double* __restrict__ eig, int n, double* __restrict__ s_out,
                                         double* __restrict__ s_prev, double* __restrict__ delta_out,
                                         int update_prev, double* __restrict__ hist = nullptr,
                                         const int* __restrict__ hist_n = nullptr, double* host_delta = nullptr,
                                         int* host_flag = nullptr, const int* dev_flag = nullptr) {
  extern __shared__ double fsm[];               // lam[n], red[33]
  double* lam = fsm; double* red = fsm + n;
  if (threadIdx.x < n) lam[threadIdx.x] = eig[threadIdx.x];
  __syncthreads();
  spectrum_finalize_body(lam, red, n, s_out, s_prev, delta_out, update_prev, hist, hist_n, host_delta, host_flag, dev_flag);
}

// Householder tridiagonalisation of a small matrix (n <= 32 NC) by ONE warp, lane l <-> columns l, l + 32 (NC = 2) of
// the full symmetric matrix in shared memory (pitch n + 1: conflict-free rows).  No block barrier inside the loop: a
// step is 0.7-1.1 us where the 1024-thread kernel above pays ~2 us for its four barriers and broadcast phases alone.
// Same reflector conventions (u = x - beta e_1, H = I - gamma u u^T, entries with |tail|^2 <= 1e-280 dropped), so d, e
// agree to rounding.  S: n (n + 1) + 2 n doubles.  All threads of the CTA load; warp 0 works; ends with a block barrier.
__host__ __device__ inline size_t tri_warp_smem_bytes(int n) { return sizeof(double) * ((size_t)n * (n + 1) + 2 * (size_t)n + 2); }
template <int NC>
__device__ __forceinline__ void tridiag_warp_body(double* S, const double* Cmat, int n, double* dvec, double* evec) {
  const int LD = n + 1;
  double* us = S + n * LD;
  double* ps = us + n;
  const int tid = threadIdx.x, lane = tid & 31;
  for (int e = tid; e < n * n; e += blockDim.x) {
    const int i = e / n, j = e - i * n;
    S[i * LD + j] = i >= j ? Cmat[(long long)i * n + j] : Cmat[(long long)j * n + i];     // lower triangle, mirrored
  }
  __syncthreads();
  if (tid < 32) {
    for (int k = 0; k < n - 2; ++k) {
      double x[NC], u[NC], p[NC];
      double t2 = 0.0;
#pragma unroll
      for (int c = 0; c < NC; ++c) {
        const int j = lane + 32 * c;
        x[c] = (j < n && j > k) ? S[k * LD + j] : 0.0;
        t2 += j > k + 1 ? x[c] * x[c] : 0.0;
      }
      const double tail2 = warp_sum(t2);
      const double alpha = S[k * LD + k + 1];
      if (!(tail2 > 1e-280)) {
        if (lane == 0) { dvec[k] = S[k * LD + k]; evec[k + 1] = alpha; }
        continue;
      }
      const double s2 = fma(alpha, alpha, tail2);
      const double sigma = s2 * rsqrt(s2);
      const double beta = alpha >= 0.0 ? -sigma : sigma;
      const double gamma = __drcp_rn(fma(-alpha, beta, s2));
#pragma unroll
      for (int c = 0; c < NC; ++c) {
        const int j = lane + 32 * c;
        u[c] = j == k + 1 ? alpha - beta : x[c];                  // 0 for j <= k and j >= n
        if (j < n) us[j] = u[c];
      }
      __syncwarp();
      double acc[NC][4];
#pragma unroll
      for (int c = 0; c < NC; ++c) acc[c][0] = acc[c][1] = acc[c][2] = acc[c][3] = 0.0;
      int jo[NC];                                                   // column offsets; lanes / columns beyond n - 1 read a
#pragma unroll                                                      // valid column (results discarded)
      for (int c = 0; c < NC; ++c) jo[c] = (lane + 32 * c < n) ? lane + 32 * c : 0;
      {
        int i = k + 1;
        for (; i + 4 <= n; i += 4) {                                // four rows in flight per column
          const double u0 = us[i], u1 = us[i + 1], u2 = us[i + 2], u3 = us[i + 3];
          const double* r0 = S + i * LD;
#pragma unroll
          for (int c = 0; c < NC; ++c) {
            acc[c][0] = fma(r0[jo[c]], u0, acc[c][0]);
            acc[c][1] = fma(r0[LD + jo[c]], u1, acc[c][1]);
            acc[c][2] = fma(r0[2 * LD + jo[c]], u2, acc[c][2]);
            acc[c][3] = fma(r0[3 * LD + jo[c]], u3, acc[c][3]);
          }
        }
        for (; i < n; ++i) {
          const double u0 = us[i];
#pragma unroll
          for (int c = 0; c < NC; ++c) acc[c][0] = fma(S[i * LD + jo[c]], u0, acc[c][0]);
        }
      }
      double pu = 0.0;
#pragma unroll
      for (int c = 0; c < NC; ++c) {
        const int j = lane + 32 * c;
        p[c] = (j < n && j > k) ? gamma * ((acc[c][0] + acc[c][1]) + (acc[c][2] + acc[c][3])) : 0.0;
        pu = fma(p[c], u[c], pu);
        if (j < n) ps[j] = p[c];
      }
      const double cf = 0.5 * gamma * warp_sum(pu);
      __syncwarp();
      {
        double aj[NC], bj[NC];
        bool on[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) {
          const int j = lane + 32 * c;
          aj[c] = fma(-2.0 * cf, u[c], p[c]); bj[c] = u[c];
          on[c] = j < n && j > k;
        }
        int i = k + 1;
        for (; i + 4 <= n; i += 4) {                                // four rows in flight per column
          const double u0 = us[i], u1 = us[i + 1], u2 = us[i + 2], u3 = us[i + 3];
          const double p0 = ps[i], p1 = ps[i + 1], p2 = ps[i + 2], p3 = ps[i + 3];
          double* r0 = S + i * LD;
#pragma unroll
          for (int c = 0; c < NC; ++c) {
            if (on[c]) {
              double* e = r0 + jo[c];
              const double v0 = e[0], v1 = e[LD], v2 = e[2 * LD], v3 = e[3 * LD];
              e[0] = fma(-p0, bj[c], fma(-u0, aj[c], v0));
              e[LD] = fma(-p1, bj[c], fma(-u1, aj[c], v1));
              e[2 * LD] = fma(-p2, bj[c], fma(-u2, aj[c], v2));
              e[3 * LD] = fma(-p3, bj[c], fma(-u3, aj[c], v3));
            }
          }
        }
        for (; i < n; ++i) {
          const double u0 = us[i], p0 = ps[i];
#pragma unroll
          for (int c = 0; c < NC; ++c)
            if (on[c]) { double* e = S + i * LD + jo[c]; e[0] = fma(-p0, bj[c], fma(-u0, aj[c], e[0])); }
        }
      }
      if (lane == 0) { dvec[k] = S[k * LD + k]; evec[k + 1] = beta; }
      __syncwarp();
    }
    if (lane == 0) {
      if (n >= 2) { dvec[n - 2] = S[(n - 2) * LD + n - 2]; evec[n - 1] = S[(n - 1) * LD + n - 2]; }
      dvec[n - 1] = S[(n - 1) * LD + n - 1];
      evec[0] = 0.0;
    }
  }
  __syncthreads();
}

// n <= 128: the matrix lives in REGISTERS.  NCG x NRG warps: warp w holds the columns j = lane + 32 (w % NCG), rows
// i = w / NCG + NRG t, t = 0..15 of the full symmetric matrix (16 doubles per thread), so the rank-2 update touches no
// shared memory but u and p, and the matrix-vector product is 16 FMAs per thread + one NRG-way combine.  Three block
// barriers per step; the reflector scalars and the two warp reductions are computed redundantly by every warp.  Same
// reflector conventions as the kernels above.  <2, 4, 16>: 256 threads, n <= 64, u of the thread's rows kept in registers
// (K8 through the API at n = 36 / 64: 70 / 103 us against 105 / 187 with the shared-memory kernels).  <4, 4, 32>: 512
// threads x 32 elements, n <= 128; (x_i, p_i) re-read from shared memory as one double2 in the update, rows and column
// groups that have been eliminated are skipped (n = 100 / 128: 254 / 325 us against 316 / 440).  A 1024-thread variant
// (64 registers per thread, 32 warps repeating the scalar chain) measured slower than tridiag_smem2_kernel.
constexpr int TRIR_MAX_N = 64, TRIR_MAX_N2 = 128;
template <int NCG, int NRG, int NE>
__global__ void __launch_bounds__(32 * NCG * NRG)
tridiag_reg_kernel(const double* __restrict__ Cmat, int n, double* __restrict__ dvec, double* __restrict__ evec) {
  constexpr int NC = 32 * NCG;                                   // columns held (>= n), NE NRG >= n rows
  constexpr bool KEEPU = NE <= 16;
  // row k (x) and p: the small variant keeps two plain arrays (its u stays in registers, and the 16-byte stride of an
  // interleaved array costs it bank conflicts on the per-lane reads); the large one reads (x_i, p_i) as one double2
  __shared__ double2 up[KEEPU ? 1 : NC];
  __shared__ double us[KEEPU ? NC : 1], pb[KEEPU ? NC : 1];
  __shared__ double part[NRG][NC];
  auto X = [&](int i) -> double& { return KEEPU ? us[i] : up[i].x; };
  auto Pv = [&](int i) -> double& { return KEEPU ? pb[i] : up[i].y; };
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int cg = warp % NCG, rg = warp / NCG;
  const int j = lane + 32 * cg;
  const bool colv = j < n;
  double a[NE];
#pragma unroll
  for (int t = 0; t < NE; ++t) {
    const int i = rg + NRG * t;
    a[t] = (colv && i < n) ? (i >= j ? Cmat[(long long)i * n + j] : Cmat[(long long)j * n + i]) : 0.0;   // lower triangle, mirrored
  }
  if (tid == 0) evec[0] = 0.0;
  for (int k = 0; k < n - 2; ++k) {
    // row k (= column k) from its owners' registers
    if (rg == k % NRG) {
      const int tk = k / NRG;
      double x = a[0];
#pragma unroll
      for (int t = 1; t < NE; ++t) x = (tk == t) ? a[t] : x;
      X(j) = (colv && j > k) ? x : 0.0;
      if (j == k) dvec[k] = x;
    }
    __syncthreads();
    double xl[NCG], t2 = 0.0;
#pragma unroll
    for (int c = 0; c < NCG; ++c) { xl[c] = X(lane + 32 * c); t2 += lane + 32 * c > k + 1 ? xl[c] * xl[c] : 0.0; }
    const double tail2 = warp_sum(t2);
    const double alpha = X(k + 1);
    if (!(tail2 > 1e-280)) {                                      // uniform: every warp reduces the same numbers
      if (tid == 0) evec[k + 1] = alpha;
      __syncthreads();                                           // up is rewritten by the next step
      continue;
    }
    const double s2 = fma(alpha, alpha, tail2);
    const double sigma = s2 * rsqrt(s2);
    const double beta = alpha >= 0.0 ? -sigma : sigma;
    const double gamma = __drcp_rn(fma(-alpha, beta, s2));
    const double u1 = alpha - beta;
    // a warp whose 32 columns have all been eliminated, and groups of four rows that have been or lie beyond n, do
    // nothing: their u, p are zero (uniform branches)
    const bool wact = KEEPU || 32 * cg + 31 > k;                   // (the small variant skips nothing: the tests cost more)
    double ui[KEEPU ? NE : 1];
    const double uj = j == k + 1 ? u1 : X(j);
    if (wact) {
      double p0 = 0.0, p1 = 0.0, p2 = 0.0, p3 = 0.0;
#pragma unroll
      for (int t = 0; t < NE; t += 4) {
        if (KEEPU || (rg + NRG * (t + 3) > k && rg + NRG * t < n)) {
          double u[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const int i = rg + NRG * (t + q);
            u[q] = i == k + 1 ? u1 : X(i);                         // x_i = 0 for i <= k and i >= n
            if (KEEPU) ui[t + q] = u[q];
          }
          p0 = fma(a[t], u[0], p0); p1 = fma(a[t + 1], u[1], p1);
          p2 = fma(a[t + 2], u[2], p2); p3 = fma(a[t + 3], u[3], p3);
        }
      }
      part[rg][j] = (p0 + p1) + (p2 + p3);
    }
    __syncthreads();
    if (rg == 0) {
      double sum = 0.0;
      if (wact) {
#pragma unroll
        for (int r = 0; r < NRG; r += 2) sum += part[r][j] + part[r + 1][j];
      }
      Pv(j) = (colv && j > k) ? gamma * sum : 0.0;
    }
    __syncthreads();
    double pu = 0.0;
#pragma unroll
    for (int c = 0; c < NCG; ++c) pu = fma(Pv(lane + 32 * c), lane + 32 * c == k + 1 ? u1 : xl[c], pu);
    const double cf = 0.5 * gamma * warp_sum(pu);
    if (wact) {
      const double pj = Pv(j);
      const double aj = fma(-2.0 * cf, uj, pj), bj = uj;         // both 0 for j <= k: columns <= k stay as they are
#pragma unroll
      for (int t = 0; t < NE; t += 4) {
        if (KEEPU || (rg + NRG * (t + 3) > k && rg + NRG * t < n)) {
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const int i = rg + NRG * (t + q);
            double u, pi;                                         // (x_i, p_i): both 0 for i <= k and i >= n
            if (KEEPU) { u = ui[t + q]; pi = pb[i]; }
            else { const double2 w = up[i]; u = i == k + 1 ? u1 : w.x; pi = w.y; }
            a[t + q] = fma(-pi, bj, fma(-u, aj, a[t + q]));
          }
        }
      }
    }
    if (tid == 0) evec[k + 1] = beta;
  }
  // the last 2 x 2 block
  {
    const int i1 = n - 1, i2 = n - 2;
#pragma unroll
    for (int t = 0; t < NE; ++t) {
      const int i = rg + NRG * t;
      if (n >= 2 && i == i2 && j == i2) dvec[i2] = a[t];
      if (n >= 2 && i == i1 && j == i2) evec[i1] = a[t];
      if (i == i1 && j == i1) dvec[i1] = a[t];
    }
  }
}

// K8 in ONE launch for small corners (n <= SPEC_FUSED_MAX_N): tridiagonalisation (one warp), multisection (32 warps,
// n / 32 rounds) and finalisation by the same CTA -- at these sizes the three launches cost more than the arithmetic.
constexpr int SPEC_FUSED_MAX_N = 24;
__host__ __device__ inline size_t spectrum_fused_smem_bytes(int n) {
  const size_t a = tri2_smem_bytes(n), b = tri_warp_smem_bytes(n);
  return (a > b ? a : b) + sizeof(double) * (5 * (size_t)n + 40);
}

__device__ __forceinline__ void
spectrum_fused_body(double* tsm, const double* Cmat, int n, double* eig_out, double* s_out, double* s_prev,
                    double* delta_out, int update_prev, double* hist, const int* hist_n, double* host_delta = nullptr,
                    int* host_flag = nullptr, const int* dev_flag = nullptr) {
  double* extra = tsm + (spectrum_fused_smem_bytes(n) - sizeof(double) * (5 * (size_t)n + 40)) / sizeof(double);
  double* dv = extra;                            // n
  double* ev = dv + n;                           // n
  double2* de = reinterpret_cast<double2*>((reinterpret_cast<uintptr_t>(ev + n) + 15) & ~static_cast<uintptr_t>(15));   // n pairs
  double* lam = reinterpret_cast<double*>(de + n);              // n
  double* red = lam + n;                         // 33
  tridiag_warp_body<1>(tsm, Cmat, n, dv, ev);
  double glo, ghi, isc;
  multisect_setup(dv, ev, n, de, red, glo, ghi, isc);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int idx = warp; idx < n; idx += (int)(blockDim.x >> 5)) {
    const double l = multisect_warp<true>(de, n, idx, glo, ghi) * isc;
    if (lane == 0) { lam[idx] = l; eig_out[idx] = l; }
  }
  __syncthreads();
  spectrum_finalize_body(lam, red, n, s_out, s_prev, delta_out, update_prev, hist, hist_n, host_delta, host_flag, dev_flag);
}

__global__ void __launch_bounds__(TRI2_NT, 1)
spectrum_fused_kernel(const double* Cmat, int n, double* eig_out, double* s_out, double* s_prev, double* delta_out,
                      int update_prev, double* hist, const int* hist_n, double* host_delta = nullptr,
                      int* host_flag = nullptr, const int* dev_flag = nullptr) {
  extern __shared__ __align__(16) double tsm[];
  spectrum_fused_body(tsm, Cmat, n, eig_out, s_out, s_prev, delta_out, update_prev, hist, hist_n, host_delta, host_flag, dev_flag);
}

}  // namespace qk
