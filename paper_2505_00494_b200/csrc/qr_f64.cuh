// K2: unpivoted Householder QR of the reduced corner c~ (rows x n, row-major,
// ld = n).  Reflector convention (LAPACK dlarfg): for a column x
// with head alpha and tail t:  sigma = ||x||, beta = -sign(alpha) sigma,
// tau = (beta - alpha)/beta, v = [1; t/(alpha - beta)], H = I - tau v v^T,
// H x = beta e_1.  R's diagonal is beta; the later sign fix makes it >= 0.
//
// Level-2 column kernels (this file, first section) are the simple correct path;
// the blocked compact-WY path (second section) uses them only inside a panel.
#pragma once
#include <cooperative_groups.h>

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


// ------------------------------------------------------------------------------
// Blocked path: panel factorisation by ONE thread-block cluster.
//
// The panel V[j0:, j0:j0+nbw] (nbw <= NB columns) is split by rows over the C
// CTAs of the cluster; every CTA keeps its slice in shared memory (or works in
// place in global/L2 when the slice does not fit).  For column k ONE reduction
// gives everything the reflector and its application inside the panel need:
//     g_j = sum_{i > r} x_i y_ij   (j = k..nbw-1; g_k = ||tail||^2),   r = j0+k,
// plus the diagonal row (alpha = x_r and y_rj) from its owner.  Partials are
// written to every CTA's shared memory through DSMEM, one cluster barrier, then
// every CTA sums them in rank order (bitwise identical everywhere, deterministic)
//     sigma = sqrt(alpha^2 + g_k), beta = -sign(alpha) sigma, tau = (beta-alpha)/beta,
//     scale = 1/(alpha-beta),  w_j = tau (y_rj + scale g_j),
//     y_ij -= (scale x_i) w_j  (i > r),   y_rj -= w_j.
// Column k is left unscaled until write-back so nobody races on it.
// Afterwards the Gram matrix of the unit-lower-trapezoidal reflectors gives the
// compact-WY factor T (forward larft recurrence), written to Tp[NB][NB].
template <int NB>
__global__ void __launch_bounds__(1024, 1)
qr_panel_cluster_kernel(double* __restrict__ V, long long ld, long long m, int j0, int nbw,
                        double* __restrict__ Vc, double* __restrict__ tau, double* __restrict__ Tp,
                        long long rpc, int use_smem) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int C = (int)cluster.num_blocks();
  const int rank = (int)cluster.block_rank();
  constexpr int NT = 1024, NRG = NT / NB, NW = NT / 32;
  extern __shared__ __align__(16) double sm[];
  // layout: exch[2][Cmax=16][NB] | rowv[2][NB] | red[NW][NB] | par[3][NB] (scale,beta,tau) | G[NB*NB] |
  //         exchG[16][NB*NB] (rank 0 uses) | slice
  double* exch = sm;
  double* rowv = exch + 2 * 16 * NB;
  double* red = rowv + 2 * NB;
  double* par = red + NW * NB;
  double* Gs = par + 3 * NB;
  double* exchG = Gs + NB * NB;
  double* slice = exchG + 16 * NB * NB;

  const int tid = threadIdx.x, col = tid % NB, rg = tid / NB, warp = tid >> 5, lane = tid & 31;
  const long long row_lo = (long long)j0 + (long long)rank * rpc;
  long long row_hi = row_lo + rpc; if (row_hi > m) row_hi = m;
  const int nloc = row_hi > row_lo ? (int)(row_hi - row_lo) : 0;
  double* pan; long long ldp;
  if (use_smem) {
    pan = slice; ldp = NB;
    for (int idx = tid; idx < nloc * NB; idx += NT) {
      int li = idx / NB, c = idx % NB;
      slice[idx] = c < nbw ? V[(row_lo + li) * ld + j0 + c] : 0.0;
    }
  } else {
    pan = V + row_lo * ld + j0; ldp = ld;
  }
  __syncthreads();
  cluster.sync();          // every CTA of the cluster is resident before the first DSMEM store

  int buf = 0;
  for (int k = 0; k < nbw; ++k) {
    const long long r = (long long)j0 + k;
    double acc = 0.0;
    if (col >= k && col < nbw) {
      for (int li = rg; li < nloc; li += NRG) {
        if (row_lo + li > r) acc = fma(pan[li * ldp + k], pan[li * ldp + col], acc);
      }
    }
    if (NB == 16) acc += __shfl_xor_sync(0xffffffffu, acc, 16);
    if (lane < NB) red[warp * NB + lane] = acc;      // NB == 32: every lane; NB == 16: lanes 0..15
    __syncthreads();
    if (tid < NB) {
      double g = 0.0;
      for (int w = 0; w < NW; ++w) g += red[w * NB + tid];
      const bool owner = (r >= row_lo && r < row_hi);
      double rv = owner ? pan[(r - row_lo) * ldp + tid] : 0.0;
      for (int q = 0; q < C; ++q) {
        double* rex = cluster.map_shared_rank(exch, q);
        rex[(buf * 16 + rank) * NB + tid] = g;
        if (owner) { double* rr = cluster.map_shared_rank(rowv, q); rr[buf * NB + tid] = rv; }
      }
    }
    cluster.sync();
    double gk = 0.0, gj = 0.0;
    for (int q = 0; q < C; ++q) { gk += exch[(buf * 16 + q) * NB + k]; gj += exch[(buf * 16 + q) * NB + col]; }
    const double alpha = rowv[buf * NB + k], yrj = rowv[buf * NB + col];
    double tk = 0.0, scale = 0.0, beta = alpha;
    if (gk > 0.0) {
      double sigma = sqrt(fma(alpha, alpha, gk));
      beta = alpha >= 0.0 ? -sigma : sigma;
      tk = (beta - alpha) / beta;
      scale = 1.0 / (alpha - beta);
    }
    if (tid == 0) { par[k] = scale; par[NB + k] = beta; par[2 * NB + k] = tk; }
    if (col > k && col < nbw && tk != 0.0) {
      const double w = tk * fma(scale, gj, yrj);
      for (int li = rg; li < nloc; li += NRG) {
        long long gi = row_lo + li;
        if (gi > r) pan[li * ldp + col] = fma(-(pan[li * ldp + k] * scale), w, pan[li * ldp + col]);
        else if (gi == r) pan[li * ldp + col] -= w;
      }
    }
    __syncthreads();
    buf ^= 1;
  }

  // write-back: in-place factor (R above/on the diagonal, scaled v below), clean reflectors Vc
  for (int idx = tid; idx < nloc * NB; idx += NT) {
    int li = idx / NB, c = idx % NB;
    if (c >= nbw) continue;
    long long gi = row_lo + li, rc = (long long)j0 + c;
    double x = pan[li * ldp + c], vout, vclean;
    if (gi > rc) { vclean = x * par[c]; vout = vclean; }
    else if (gi == rc) { vclean = 1.0; vout = par[NB + c]; }
    else { vclean = 0.0; vout = x; }
    V[gi * ld + j0 + c] = vout;
    Vc[gi * ld + j0 + c] = vclean;
    if (use_smem) slice[idx] = vclean;
  }
  if (rank == 0 && tid < nbw) tau[j0 + tid] = par[2 * NB + tid];
  __syncthreads();

  // Gram of the clean reflectors (strict upper part is what larft needs)
  {
    constexpr int NP = NB * NB, NQ = NT / NP > 0 ? NT / NP : 1;   // NB=16: 256 pairs x 4 row subsets
    const int pidx = tid % NP, a = pidx / NB, c = pidx % NB, qs = tid / NP;
    double g = 0.0;
    const double* gsrc = use_smem ? slice : Vc + row_lo * ld + j0;
    const long long gld = use_smem ? NB : ld;
    if (tid < NP * NQ && a < c && c < nbw) {
      for (int li = qs; li < nloc; li += NQ) g = fma(gsrc[li * gld + a], gsrc[li * gld + c], g);
    }
    // reduce the NQ row subsets through scratch behind the slice (exchG receives remote writes)
    __syncthreads();
    double* scratch = slice + (use_smem ? (size_t)rpc * NB : 0);    // NQ*NP doubles reserved by the host
    if (tid < NP * NQ) scratch[qs * NP + pidx] = g;
    __syncthreads();
    if (tid < NP) {
      double t = 0.0;
      for (int q = 0; q < NQ; ++q) t += scratch[q * NP + tid];
      double* rg0 = cluster.map_shared_rank(exchG, 0);
      rg0[rank * NP + tid] = t;
    }
  }
  cluster.sync();
  if (rank == 0) {
    constexpr int NP = NB * NB;
    if (tid < NP) {
      double t = 0.0;
      for (int q = 0; q < C; ++q) t += exchG[q * NP + tid];
      Gs[tid] = t;
    }
    __syncthreads();
    if (tid < NB) {                 // lane a builds row a of T (upper triangular), columns left to right
      const int a = tid;
      double Trow[NB];
#pragma unroll
      for (int i = 0; i < NB; ++i) Trow[i] = 0.0;
#pragma unroll
      for (int i = 0; i < NB; ++i) {
        if (i < nbw) {
          double ti = par[2 * NB + i];
          if (a == i) Trow[i] = ti;
          else if (a < i) {
            double s = 0.0;
#pragma unroll
            for (int c = 0; c < NB; ++c)
              if (c >= a && c < i) s = fma(Trow[c], Gs[c * NB + i], s);
            Trow[i] = -ti * s;
          }
        }
      }
#pragma unroll
      for (int i = 0; i < NB; ++i) Tp[a * NB + i] = Trow[i];
    }
  }
}

}  // namespace qk
