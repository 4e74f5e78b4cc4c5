// Whole-iteration kernels for tiny problems: when C, T, c~, Q, a and both m x m
// intermediates fit in ONE CTA's shared memory (cfg0: d = 2, D = 2, chi = 8, m = 32), K1..K6 run as one launch
// (small_front_kernel) and K7 as one more (small_k7_kernel) instead of ~18 launches of a few microseconds each.
// Plain DFMA loops over shared memory -- at these sizes the step is launch-latency-bound, not a tensor-core problem.
// Same equations and the same Householder QR (dlarfg convention, then diag(R) >= 0) as the large path:
//   (E1) X[(j,u),k] = sum_i C[j,i] T[i,u,k]
//   (E2) X = Q R
//   (E3) P[(u,l),(J,m)] = sum_j Q[(j,u),m] T[j,l,J];  S[(J,d),(m,r)] = sum_(u,l) P[(u,l),(J,m)] a[(u,l),(d,r)];
//        T'[(m,r),n] = sum_(J,d) S[(J,d),(m,r)] Q[(J,d),n]
//   (E4) W[(m,r),n] = sum_k R[m,k] Q[(k,r),n];  C'[p,n] = sum_(m,r) T'[(m,r),p] W[(m,r),n]
// Deterministic (fixed summation orders).
#pragma once
#include "kernels_misc.cuh"
#include "spectrum.cuh"

namespace qk {

constexpr int SMALL_NT = 1024;       // = TRI2_NT: the fused run kernel calls the K8 body, written for 32 warps

__host__ __device__ inline size_t small_front_doubles(int b, int chi) {
  const size_t m = (size_t)b * chi, b2 = (size_t)b * b;
  return (size_t)chi * chi * 2 + m * chi * 5 + b2 * b2 + 2 * m * m + 2 * chi + 64;
}

// Inputs (global): C[chi][chi], T[chi][b][chi], a_mat[b*b][lda].  Outputs (global): X, Q (m x chi), R (chi x chi),
// Tn (m x chi), Cn (chi x chi) -- the un-normalised C', T' that K7 consumes.
// (no __restrict__ on the bodies: small_run_kernel calls them in a loop in which C, T are rewritten by the K7 body, so
// their loads must not go through the non-coherent read-only path)
// Householder QR of a tiny c~ (chi <= 8 columns, m <= 32 RPL rows) by ONE warp: lane l holds the rows l + 32 r in registers,
// no block barrier per column, the dot products of a reflector with all columns are reduced together.  Same reflectors
// (dlarfg convention) and sign fix (diag(R) >= 0) as the column loop in small_front_body.  X (m x chi) -> Q, R, all in
// shared memory.
template <int RPL>
__device__ __forceinline__ void small_qr_warp(const double* X, double* Q, double* R, int m, int chi, int lane) {
  double x[RPL][8], q[RPL][8], tauv[8];
#pragma unroll
  for (int r = 0; r < RPL; ++r)
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const int i = lane + 32 * r;
      x[r][c] = (i < m && c < chi) ? X[i * chi + c] : 0.0;
      q[r][c] = (i == c) ? 1.0 : 0.0;
    }
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    tauv[k] = 0.0;
    if (k < chi) {
      double acc = 0.0;
#pragma unroll
      for (int r = 0; r < RPL; ++r) { const int i = lane + 32 * r; if (i > k) acc = fma(x[r][k], x[r][k], acc); }
      const double tail2 = warp_sum(acc);
      const double alpha = __shfl_sync(0xffffffffu, x[0][k], k);
      double t = 0.0, scale = 0.0, beta = alpha;
      if (tail2 > 0.0) {                                            // one rsqrt and two independent reciprocals instead of
        const double s2 = fma(alpha, alpha, tail2);                 // sqrt and two divisions (~250 cycles less per column)
        const double sigma = s2 * rsqrt(s2);
        beta = alpha >= 0.0 ? -sigma : sigma;
        t = (beta - alpha) * __drcp_rn(beta);
        scale = __drcp_rn(alpha - beta);
      }
      double v[RPL];
#pragma unroll
      for (int r = 0; r < RPL; ++r) {
        const int i = lane + 32 * r;
        v[r] = i > k ? x[r][k] * scale : (i == k ? 1.0 : 0.0);
        x[r][k] = i > k ? v[r] : (i == k ? beta : x[r][k]);          // reflector below the diagonal, R on and above it
      }
      tauv[k] = t;
      if (t != 0.0) {
        double d[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) { double acc2 = 0.0;
          if (c > k) {
#pragma unroll
            for (int r = 0; r < RPL; ++r) acc2 = fma(v[r], x[r][c], acc2);
          }
          d[c] = acc2; }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
#pragma unroll
          for (int c = 0; c < 8; ++c) if (c > k) d[c] += __shfl_xor_sync(0xffffffffu, d[c], o);
#pragma unroll
        for (int c = 0; c < 8; ++c)
          if (c > k) {
            const double w = t * d[c];
#pragma unroll
            for (int r = 0; r < RPL; ++r) x[r][c] = fma(-v[r], w, x[r][c]);
          }
      }
    }
  }
#pragma unroll
  for (int k = 7; k >= 0; --k) {                                  // Q = H_0 ... H_{chi-1} [I; 0]
    if (k < chi && tauv[k] != 0.0) {
      double v[RPL];
#pragma unroll
      for (int r = 0; r < RPL; ++r) { const int i = lane + 32 * r; v[r] = i > k ? x[r][k] : (i == k ? 1.0 : 0.0); }
      double d[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) { double acc2 = 0.0;
        if (c >= k) {
#pragma unroll
          for (int r = 0; r < RPL; ++r) acc2 = fma(v[r], q[r][c], acc2);
        }
        d[c] = acc2; }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int c = 0; c < 8; ++c) if (c >= k) d[c] += __shfl_xor_sync(0xffffffffu, d[c], o);
#pragma unroll
      for (int c = 0; c < 8; ++c)
        if (c >= k) {
          const double w = tauv[k] * d[c];
#pragma unroll
          for (int r = 0; r < RPL; ++r) q[r][c] = fma(-v[r], w, q[r][c]);
        }
    }
  }
  // sign fix: diag(R) >= 0; R's row k is held by lane k (k < 8 <= 32)
  double sg[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) sg[c] = __shfl_sync(0xffffffffu, x[0][c], c) < 0.0 ? -1.0 : 1.0;
  double mys = 1.0;
#pragma unroll
  for (int c = 0; c < 8; ++c) mys = lane == c ? sg[c] : mys;
#pragma unroll
  for (int r = 0; r < RPL; ++r)
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const int i = lane + 32 * r;
      if (i < m && c < chi) Q[i * chi + c] = q[r][c] * sg[c];
    }
  if (lane < chi) {
#pragma unroll
    for (int c = 0; c < 8; ++c) if (c < chi) R[lane * chi + c] = c >= lane ? x[0][c] * mys : 0.0;
  }
}

template <int NT>
__device__ __forceinline__ void
small_front_body(double* ssm, const double* Cg, const double* Tg, const double* ag,
                 long long lda, int b, int chi, double* Xg, double* Qg, double* Rg, double* Tng, double* Cng) {
  const int m = b * chi, b2 = b * b, mc = m * chi, cc = chi * chi;
  double* C = ssm;                 // chi^2
  double* R = C + cc;              // chi^2
  double* T = R + cc;              // m chi    T[i][u][k]
  double* X = T + mc;              // m chi    c~, then the reflectors V (below the diagonal) and R (upper)
  double* Q = X + mc;              // m chi
  double* Tn = Q + mc;             // m chi
  double* W = Tn + mc;             // m chi
  double* a = W + mc;              // b^4      a[(u,l)][(d,r)]
  double* P = a + (size_t)b2 * b2; // m^2      P[(u,l)][(J,m)]
  double* S = P + (size_t)m * m;   // m^2      S[(J,d)][(m,r)]
  double* tau = S + (size_t)m * m; // chi
  double* wv = tau + chi;          // chi + 64 scratch
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = NT / 32;

  for (int i = tid; i < cc; i += NT) C[i] = Cg[i];
  for (int i = tid; i < mc; i += NT) T[i] = Tg[i];
  for (int i = tid; i < b2 * b2; i += NT) a[i] = ag[(long long)(i / b2) * lda + i % b2];
  __syncthreads();
  // (E1) X[(j,u),k]: row (j,u) = j*b+u; T as chi x (b chi) row-major: T[i][(u,k)]
  for (int o = tid; o < mc; o += NT) {
    const int j = o / (b * chi), uk = o % (b * chi);
    double s = 0.0;
    for (int i = 0; i < chi; ++i) s = fma(C[j * chi + i], T[i * b * chi + uk], s);
    X[o] = s;                                            // o = (j*b+u)*chi + k
  }
  __syncthreads();
  for (int i = tid; i < mc; i += NT) Xg[i] = X[i];
  // (E2) Householder QR: by one warp in registers where the matrix is small enough (small_qr_warp), else column by column
  if (chi <= 8 && m <= (NT <= 256 ? 96 : 32)) {       // (the 1024-thread kernels have 64 registers per thread: one row per lane)
    if (warp == 0) {
      if (m <= 32) small_qr_warp<1>(X, Q, R, m, chi, lane);
      else if (NT <= 256) small_qr_warp<3>(X, Q, R, m, chi, lane);
    }
    __syncthreads();
  } else {
    // (E2) Householder QR, column by column: warp 0 forms the reflector, then one warp per remaining column applies it
    for (int k = 0; k < chi; ++k) {
      if (warp == 0) {
        double acc = 0.0;
        for (int i = k + 1 + lane; i < m; i += 32) { const double x = X[i * chi + k]; acc = fma(x, x, acc); }
        const double tail2 = warp_sum(acc);
        const double alpha = X[k * chi + k];
        double t = 0.0, scale = 0.0, beta = alpha;
        if (tail2 > 0.0) {
          const double sigma = sqrt(fma(alpha, alpha, tail2));
          beta = alpha >= 0.0 ? -sigma : sigma;
          t = (beta - alpha) / beta;
          scale = 1.0 / (alpha - beta);
        }
        __syncwarp();
        for (int i = k + 1 + lane; i < m; i += 32) X[i * chi + k] *= scale;
        if (lane == 0) { X[k * chi + k] = beta; tau[k] = t; }
      }
      __syncthreads();
      const double t = tau[k];
      if (t != 0.0) {
        for (int j = k + 1 + warp; j < chi; j += NW) {
          double acc = 0.0;
          for (int i = k + lane; i < m; i += 32) acc = fma(i == k ? 1.0 : X[i * chi + k], X[i * chi + j], acc);
          const double w = t * warp_sum(acc);
          for (int i = k + lane; i < m; i += 32) X[i * chi + j] = fma(-(i == k ? 1.0 : X[i * chi + k]), w, X[i * chi + j]);
        }
      }
      __syncthreads();
    }
    for (int o = tid; o < cc; o += NT) R[o] = (o % chi >= o / chi) ? X[o] : 0.0;      // X's top chi rows
    for (int o = tid; o < mc; o += NT) Q[o] = (o / chi == o % chi) ? 1.0 : 0.0;
    __syncthreads();
    for (int k = chi - 1; k >= 0; --k) {                   // Q = H_0 ... H_{chi-1} [I; 0]
      const double t = tau[k];
      if (t != 0.0) {
        for (int j = k + warp; j < chi; j += NW) {
          double acc = 0.0;
          for (int i = k + lane; i < m; i += 32) acc = fma(i == k ? 1.0 : X[i * chi + k], Q[i * chi + j], acc);
          const double w = t * warp_sum(acc);
          for (int i = k + lane; i < m; i += 32) Q[i * chi + j] = fma(-(i == k ? 1.0 : X[i * chi + k]), w, Q[i * chi + j]);
        }
      }
      __syncthreads();
    }
    if (tid < chi) wv[tid] = R[tid * chi + tid] < 0.0 ? -1.0 : 1.0;                         // sign fix: diag(R) >= 0
    __syncthreads();
    for (int o = tid; o < mc; o += NT) Q[o] *= wv[o % chi];
    for (int o = tid; o < cc; o += NT) R[o] *= wv[o / chi];
    __syncthreads();
  }
  for (int o = tid; o < mc; o += NT) Qg[o] = Q[o];
  for (int o = tid; o < cc; o += NT) Rg[o] = R[o];
  // (E3a) P[(u,l),(J,mm)] = sum_j Q[(j,u),mm] T[j,l,J]
  for (int o = tid; o < m * m; o += NT) {
    const int ul = o / cc, Jm = o % cc, u = ul / b, l = ul % b, J = Jm / chi, mm = Jm % chi;
    double s = 0.0;
    for (int j = 0; j < chi; ++j) s = fma(Q[(j * b + u) * chi + mm], T[(j * b + l) * chi + J], s);
    P[o] = s;
  }
  __syncthreads();
  // (E3b) S[(J,d),(mm,r)] = sum_(u,l) P[(u,l),(J,mm)] a[(u,l),(d,r)]
  for (int o = tid; o < m * m; o += NT) {
    const int Jd = o / m, mr = o % m, J = Jd / b, d = Jd % b, mm = mr / b, r = mr % b;
    double s = 0.0;
    for (int ul = 0; ul < b2; ++ul) s = fma(P[ul * cc + J * chi + mm], a[ul * b2 + d * b + r], s);
    S[o] = s;
  }
  __syncthreads();
  // (E3c) T'[(mm,r),n] = sum_(J,d) S[(J,d),(mm,r)] Q[(J,d),n];   (E4a) W[(mm,r),n] = sum_k R[mm,k] Q[(k,r),n]
  for (int o = tid; o < mc; o += NT) {
    const int mr = o / chi, n = o % chi, mm = mr / b, r = mr % b;
    double s = 0.0;
    for (int Jd = 0; Jd < m; ++Jd) s = fma(S[Jd * m + mr], Q[Jd * chi + n], s);
    Tn[o] = s;
    double w = 0.0;
    for (int k = mm; k < chi; ++k) w = fma(R[mm * chi + k], Q[(k * b + r) * chi + n], w);    // R upper triangular
    W[o] = w;
  }
  __syncthreads();
  for (int o = tid; o < mc; o += NT) Tng[o] = Tn[o];
  // (E4b) C'[p,n] = sum_(mm,r) T'[(mm,r),p] W[(mm,r),n]
  for (int o = tid; o < cc; o += NT) {
    const int p = o / chi, n = o % chi;
    double s = 0.0;
    for (int mr = 0; mr < m; ++mr) s = fma(Tn[mr * chi + p], W[mr * chi + n], s);
    Cng[o] = s;
  }
}

constexpr int SMALL_NT1 = 256;        // stand-alone kernels at the smallest sizes (m <= 40): fewer warps, cheaper barriers
template <int NT>
__global__ void __launch_bounds__(NT, 1)
small_front_kernel(const double* Cg, const double* Tg, const double* ag, long long lda, int b, int chi, double* Xg,
                   double* Qg, double* Rg, double* Tng, double* Cng) {
  extern __shared__ __align__(16) double ssm[];
  small_front_body<NT>(ssm, Cg, Tg, ag, lda, b, chi, Xg, Qg, Rg, Tng, Cng);
}

// K7 in one CTA: C, T <- sym(C', T') / ||.||_F, the NaN / zero-norm flag, the norms and (hist != null) the history record.
template <int NT>
__device__ __forceinline__ void
small_k7_body(const double* Cn, const double* Tn, int chi, int b, int symmetrize, double* C, double* T, double* scal,
              int* flag, double* hist, int* hist_n, const double* R) {
  __shared__ double sh[33];
  const int tid = threadIdx.x;
  const int cc = chi * chi, bc = b * chi, mc = bc * chi;
  double ac = 0.0, at = 0.0;
  for (int o = tid; o < cc; o += NT) {
    double v = Cn[o];
    if (symmetrize) v = 0.5 * (v + Cn[(o % chi) * chi + o / chi]);
    C[o] = v; ac = fma(v, v, ac);
  }
  for (int o = tid; o < mc; o += NT) {
    const int i = o / bc, s = (o / chi) % b, k = o % chi;
    double v = Tn[o];
    if (symmetrize) v = 0.5 * (v + Tn[k * bc + s * chi + i]);
    T[o] = v; at = fma(v, v, at);
  }
  const double nc = sqrt(block_sum(ac, sh)), nt = sqrt(block_sum(at, sh));
  double ratio = 0.0;
  if (hist) {
    double mn = INFINITY, mx = -INFINITY;
    for (int k = tid; k < chi; k += NT) { const double v = R[k * chi + k]; mn = fmin(mn, v); mx = fmax(mx, v); }
    const double gmx = block_max(mx, sh), gmn = -block_max(-mn, sh);
    ratio = gmx != 0.0 ? gmn / gmx : 0.0;
  }
  __syncthreads();                                       // every thread's own C, T elements are written; same thread rescales them
  for (int o = tid; o < cc; o += NT) C[o] = C[o] / nc;
  for (int o = tid; o < mc; o += NT) T[o] = T[o] / nt;
  if (tid == 0) {
    scal[0] = nc; scal[1] = nt;
    if (!(nc > 0.0) || !(nt > 0.0) || isinf(nc) || isinf(nt)) *flag = 1;
    if (hist) {
      const int idx = *hist_n;
      double* rec = hist + (size_t)(idx % QRCTM_HIST_CAP) * 4;
      rec[0] = __longlong_as_double(0x7ff8000000000000LL); rec[1] = nc; rec[2] = nt; rec[3] = ratio;
      *hist_n = idx + 1;
    }
  }
}

__global__ void __launch_bounds__(SMALL_NT1, 1)
small_k7_kernel(const double* Cn, const double* Tn, int chi, int b, int symmetrize, double* C, double* T, double* scal,
                int* flag, double* hist, int* hist_n, const double* R) {
  small_k7_body<SMALL_NT1>(Cn, Tn, chi, b, symmetrize, C, T, scal, flag, hist, hist_n, R);
}

// K9 for tiny problems: the whole run(max_iter, tol) loop in ONE launch of one CTA -- K1..K6, K7, and every
// check_every steps K8 with the convergence decision delta < tol taken on the device; no host round trip per
// iteration.  Same semantics as the host drivers (iters = steps executed, delta = last delta or +inf).
// out[0] = iterations done, out[1] = last delta (doubles, global).
__host__ __device__ inline size_t small_run_smem_bytes(int b, int chi) {
  const size_t f = sizeof(double) * small_front_doubles(b, chi), k8 = spectrum_fused_smem_bytes(chi);
  return f > k8 ? f : k8;
}

__global__ void __launch_bounds__(SMALL_NT, 1)
small_run_kernel(double* C, double* T, const double* ag, long long lda, int b, int chi, int symmetrize, double* Xg,
                 double* Qg, double* Rg, double* Tng, double* Cng, double* scal, int* flag, double* hist, int* hist_n,
                 double* eig, double* s_out, double* s_prev, double* delta_out, int need_s0, int max_iter, double tol,
                 int check_every, double* out) {
  extern __shared__ __align__(16) double dyn[];
  if (need_s0) {                                 // previous spectrum = spectrum of the environment just set
    spectrum_fused_body(dyn, C, chi, eig, s_out, s_prev, delta_out, 1, nullptr, nullptr);
    __syncthreads();
  }
  double delta = INFINITY;
  int it = 1;
  for (; it <= max_iter; ++it) {
    small_front_body<SMALL_NT>(dyn, C, T, ag, lda, b, chi, Xg, Qg, Rg, Tng, Cng);
    __syncthreads();
    small_k7_body<SMALL_NT>(Cng, Tng, chi, b, symmetrize, C, T, scal, flag, hist, hist_n, Rg);
    __syncthreads();
    if (*flag) break;                            // NaN / zero norm: the host reports it
    if (it % check_every == 0 || it == max_iter) {
      spectrum_fused_body(dyn, C, chi, eig, s_out, s_prev, delta_out, 1, hist, hist_n);
      __syncthreads();
      delta = delta_out[0];
      if (delta < tol) break;
    }
  }
  if (threadIdx.x == 0) { out[0] = (double)(it <= max_iter ? it : max_iter); out[1] = delta; }
}

}  // namespace qk
