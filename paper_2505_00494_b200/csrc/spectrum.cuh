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
constexpr int TRI2_NT = 1024, TRI2_NA = 256, TRI2_NWA = TRI2_NA / 32, TRI2_MAX_N = 232;
__host__ __device__ inline size_t tri2_smem_bytes(int n) {
  return sizeof(double) * ((size_t)n * (n + 1) / 2 + 1 + 4 * (size_t)n + 16 + 8);
}

// 1024 threads.  Threads 0..255 ("group A", one per column) compute the reflector and p = gamma A u; all 32 warps
// share the rank-2 update: warp w owns the 32 columns of group w & 7 and the rows congruent to (w >> 3) modulo 4
// below them, so a column's dependent load-FMA-store chain is split four ways and unrolled four deep.
__global__ void __launch_bounds__(TRI2_NT, 1)
tridiag_smem2_kernel(const double* __restrict__ Cmat, int n, double* __restrict__ dvec, double* __restrict__ evec,
                     long long* __restrict__ prof /* null, or 8 cycle counters of the phases (thread 0) */) {
  extern __shared__ __align__(16) double tsm[];
  // (u_i, p_i) pairs, double-buffered over the steps: u = column k of the matrix (written by the thread that owns the
  // column while it updates it in the step before), p = gamma A u (written by thread i in the matrix-vector phase)
  double2* up0 = reinterpret_cast<double2*>(tsm);               // 2 x n pairs
  double* red = tsm + 4 * n;                                    // 8: per-warp partial sums of p.u
  double* sc = red + 8;                                         // 8: [0] gamma of this step (0: nothing to eliminate)
  double* L = sc + 8;                                           // n(n+1)/2
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
  const int cg = warp & 7, rph = warp >> 3;     // column group, row phase (rph = 0: group A)
  const int j = cg * 32 + lane, tj = tri_off(j);               // my column; start of my row
  const int jlo = cg * 32, jhi = jlo + 32 < n ? jlo + 32 : n;  // the columns of my warp
  const double* Lj = L + tj;                    // my row: element (j, i), i <= j
  double* Lc = L + j;                           // my column: element (i, j) at Lc[tri(i)], i >= j
  for (int k = 0; k < n - 2; ++k) {
    double2* up = up0 + (k & 1) * n;
    double2* upn = up0 + ((k + 1) & 1) * n;
    const bool active = j > k && j < n;
    const bool wact = jlo < n && jhi > k + 1;    // warp-uniform: some lane of this warp is active
    if (rph == 0) {
      // ---- reflector of column k (rows k+1 .. n-1), redundantly in every warp of group A
      double acc = 0.0;
      for (int i = k + 2 + lane; i < n; i += 32) { const double x = up[i].x; acc = fma(x, x, acc); }
      const double tail2 = warp_sum(acc);
      const double alpha = up[k + 1].x;
      if (tid == 0) dvec[k] = L[tri_off(k) + k];
      // nothing to eliminate: H = I.  Entries below 1e-140 in magnitude are dropped rather than eliminated: gamma ~
      // 1 / tail2 would overflow, and the perturbation is 120 orders below rounding for ||C|| ~ 1
      if (!(tail2 > 1e-280)) {
        if (tid == 0) { evec[k + 1] = alpha; sc[0] = 0.0; }
        for (int i = k + 2 + tid; i < n; i += TRI2_NA) upn[i].x = L[tri_off(i) + k + 1];
      } else {
        const double s2 = fma(alpha, alpha, tail2);
        const double sigma = s2 * rsqrt(s2);                     // 1-2 ulp: only perturbs e_{k+1} at rounding level
        const double beta = alpha >= 0.0 ? -sigma : sigma;
        const double u1 = alpha - beta;
        const double gamma = __drcp_rn(fma(-alpha, beta, s2));   // 1 / (beta (beta - alpha)),  beta^2 = s2
        if (tid == 0) { evec[k + 1] = beta; sc[0] = gamma; }
        TRI_TICK(1);
        // ---- p_j = gamma sum_{i > k} A_sym[i][j] u_i for my column: rows above my warp's columns come from my row
        // (per-lane base + uniform offset), rows below them from my column (uniform row start + lane), the <= 32
        // rows in between are mixed
        double uj = 0.0, pj = 0.0;
        if (wact) {
          const int jc = active ? j : (k + 1 > jlo ? k + 1 : jlo);  // inactive lanes compute a valid column (discarded)
          const double* Ljc = active ? Lj : L + tri_off(jc);
          const double* Lcc = L + jc;
          uj = (jc == k + 1) ? u1 : up[jc].x;
          double a0 = Ljc[k + 1] * u1, a1 = 0.0;                  // i = k+1: element (jc, k+1)
          int i = k + 2;
          const int e1 = jlo < n ? jlo : n;
          for (; i + 2 <= e1; i += 2) {                           // rows above the warp's columns: my row
            a0 = fma(Ljc[i], up[i].x, a0);
            a1 = fma(Ljc[i + 1], up[i + 1].x, a1);
          }
          int off = tri_off(i);
          for (; i < jhi; ++i) {                                  // mixed rows
            a0 = fma(i < jc ? Ljc[i] : Lcc[off], up[i].x, a0);
            off += i + 1;
          }
          for (; i + 2 <= n; i += 2) {                            // rows below: my column
            a0 = fma(Lcc[off], up[i].x, a0);
            a1 = fma(Lcc[off + i + 1], up[i + 1].x, a1);
            off += 2 * i + 3;
          }
          if (i < n) a0 = fma(Lcc[off], up[i].x, a0);
          pj = active ? gamma * (a0 + a1) : 0.0;
          if (active) up[j] = make_double2(uj, pj); else uj = 0.0;   // (u_{k+1} = u1 replaces the raw column entry)
        }
        const double q = warp_sum(pj * uj);
        if (lane == 0) red[warp] = q;
      }
    }
    TRI_TICK(2);
    __syncthreads();
    TRI_TICK(3);
    const double gamma = sc[0];
    // ---- A -= u w^T + w u^T: x = A_ij - u_i (p_j - 2 cf u_j) - p_i u_j,  cf = (gamma/2) p.u
    if (gamma != 0.0 && wact && active) {
      double pu = 0.0;
#pragma unroll
      for (int w = 0; w < TRI2_NWA; ++w) pu += red[w];
      const double cf = 0.5 * gamma * pu;
      const double2 mine = up[j];
      const double aj = fma(-2.0 * cf, mine.x, mine.y), bj = mine.x;
      const bool nxt = j == k + 1;                              // my column is the next u
      const int ib = (jlo > k + 1 ? jlo : k + 1) + rph;         // warp-uniform first row of my phase; lanes join at i >= j
      for (int i = ib; i < n; i += 16) {
        double2 u[4]; double y[4]; int o[4]; bool ok[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          const int ii = i + 4 * r;
          ok[r] = ii < n && ii >= j;
          o[r] = tri_off(ok[r] ? ii : j);
          u[r] = up[ok[r] ? ii : j];
          y[r] = Lc[o[r]];
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) y[r] = fma(-u[r].y, bj, fma(-u[r].x, aj, y[r]));
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          if (ok[r]) {
            Lc[o[r]] = y[r];
            if (nxt) upn[i + 4 * r].x = y[r];
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

// Sturm count without divisions: number of eigenvalues < x of the tridiagonal whose SCALED entries (all magnitudes
// <= ~2) are de[i] = (d_i, e_i^2), from the sign changes of the leading principal minors
//   p_i = (d_i - x) p_{i-1} - e_i^2 p_{i-2}
// (q_i = p_i / p_{i-1} is the pivot sequence of sturm_count above: q_i < 0 <=> p_i and p_{i-1} differ in sign).  The
// dependent chain is one FMA per row instead of one FP64 division (~15x shorter).  Every computed p_i is the exact
// minor of a matrix with relatively perturbed entries (backward stable); only signs are used, so p is renormalised by
// an exact power of two every 4 rows (magnitudes then stay within 2^+-600 of 1).  d_i - x == 0 is replaced by 2^-100
// (a perturbation of x far below rounding at this scaling); an exact zero minor counts as a sign change.
__device__ __forceinline__ int sturm_count_minors(const double2* __restrict__ de, int n, double x) {
  double p0 = 1.0;
  double t = de[0].x - x;
  t = (t == 0.0) ? 0x1p-100 : t;
  double p1 = t;
  int neg1 = p1 < 0.0;                         // sign of p_{i-1} as used by the count (zero: opposite to its predecessor)
  int cnt = neg1;
  int i = 1;
  for (; i + 4 <= n; i += 4) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const double2 v = de[i + u];
      double tt = v.x - x;
      tt = (tt == 0.0) ? 0x1p-100 : tt;
      const double pn = fma(tt, p1, -v.y * p0);
      const int negn = (pn == 0.0) ? !neg1 : (pn < 0.0);
      cnt += negn != neg1;
      neg1 = negn; p0 = p1; p1 = pn;
    }
    // renormalise by 2^-e, e = exponent of max(|p0|, |p1|)
    const double m = fmax(fabs(p0), fabs(p1));
    const int e = ((__double2hiint(m) >> 20) & 0x7ff) - 1023;
    if (e > 64 || e < -64) {
      if (m == 0.0) { p1 = neg1 ? -1.0 : 1.0; }                         // decoupled block: restart the sequence
      else {
        const int ee = e > 1000 ? 1000 : (e < -1000 ? -1000 : e);
        const double sc = __hiloint2double((1023 - ee) << 20, 0);
        p0 *= sc; p1 *= sc;
      }
    }
  }
  for (; i < n; ++i) {
    const double2 v = de[i];
    double tt = v.x - x;
    tt = (tt == 0.0) ? 0x1p-100 : tt;
    const double pn = fma(tt, p1, -v.y * p0);
    const int negn = (pn == 0.0) ? !neg1 : (pn < 0.0);
    cnt += negn != neg1;
    neg1 = negn; p0 = p1; p1 = pn;
  }
  return cnt;
}

// Eigenvalues of the tridiagonal by warp-multisection: warp w of block B finds
// eigenvalue number idx = 8 B + w (ascending; see `ke` for the partial mode).  Each iteration the 32 lanes evaluate
// the Sturm count at 32 interior points of [a, b], shrinking the bracket 33-fold
// (about 11 iterations to the last ulp instead of ~55 bisection steps).
__global__ void __launch_bounds__(256)
multisect_kernel(const double* __restrict__ dvec, const double* __restrict__ evec, int n,
                 double* __restrict__ eig_out, int ke = 0) {
  extern __shared__ __align__(16) double msm[];               // de[n] = (d_i, e_i^2) scaled, red[33]
  double2* de = reinterpret_cast<double2*>(msm); double* red = msm + 2 * n;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  double lo = INFINITY, hi = -INFINITY;
  for (int i = tid; i < n; i += blockDim.x) {                  // Gershgorin bounds
    const double el = i > 0 ? fabs(evec[i]) : 0.0, er = i + 1 < n ? fabs(evec[i + 1]) : 0.0, di = dvec[i];
    lo = fmin(lo, di - el - er);
    hi = fmax(hi, di + el + er);
  }
  double ghi = block_max(hi, red);
  double glo = -block_max(-lo, red);
  const double bnd = fmax(fabs(glo), fabs(ghi));
  // scale the problem by an exact power of two so that every entry has magnitude <= 1 (the minors recurrence of
  // sturm_count_minors then grows by at most ~2.5 per row); eigenvalues are scaled back at the end
  int ex = 0;
  if (bnd > 0.0 && bnd < INFINITY) { frexp(bnd, &ex); }
  ex = ex > 1000 ? 1000 : (ex < -1000 ? -1000 : ex);
  const double sc = ldexp(1.0, -ex), isc = ldexp(1.0, ex);
  for (int i = tid; i < n; i += blockDim.x) {
    const double e = i > 0 ? evec[i] * sc : 0.0;
    de[i] = make_double2(dvec[i] * sc, e * e);
  }
  __syncthreads();
  glo *= sc; ghi *= sc;
  const double bs = fmax(fabs(glo), fabs(ghi));
  glo -= 2.0 * 2.220446049250313e-16 * bs * n + 0x1p-90;
  ghi += 2.0 * 2.220446049250313e-16 * bs * n + 0x1p-90;
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
    int cnt = inside ? sturm_count_minors(de, n, x) : (x >= b ? n : 0);
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
  if (lane == 0) eig_out[slot] = 0.5 * (a + b) * isc;
}

// One block, blockDim.x >= n: s = sorted |eig| (descending), delta vs s_prev.
__global__ void spectrum_finalize_kernel(const double* __restrict__ eig, int n, double* __restrict__ s_out,
                                         double* __restrict__ s_prev, double* __restrict__ delta_out,
                                         int update_prev, double* __restrict__ hist = nullptr,
                                         const int* __restrict__ hist_n = nullptr) {
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
  if (tid == 0) {
    delta_out[0] = dmax;
    if (hist && update_prev && *hist_n > 0) hist[(size_t)((*hist_n - 1) % 4096) * 4] = dmax;   // this step's record
  }
  __syncthreads();
  if (update_prev && tid < n) s_prev[tid] = s_out[tid];
}

}  // namespace qk
