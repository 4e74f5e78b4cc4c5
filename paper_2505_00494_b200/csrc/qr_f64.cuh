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
template <int NB, bool SMEM>
__global__ void __launch_bounds__(1024, 1)
qr_panel_cluster_kernel(double* __restrict__ V, long long ld, long long m, int j0, int nbw,
                        double* __restrict__ Vc, double* __restrict__ tau, double* __restrict__ Tp,
                        long long rpc) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int C = (int)cluster.num_blocks();
  const int rank = (int)cluster.block_rank();
  constexpr int NT = 1024, NRG = NT / NB, NW = NT / 32, NP = NB * NB, NQ = NT / NP > 0 ? NT / NP : 1;
  extern __shared__ __align__(16) double sm[];
  // exch[2][16][NB] | rowv[2][NB] | red[NW][NB] | par[3][NB] (scale,beta,tau) | wv[NB+1] | G[NP] |
  // exchG[16][NP] | scratch[NQ*NP] | slice
  double* exch = sm;
  double* rowv = exch + 2 * 16 * NB;
  double* red = rowv + 2 * NB;
  double* par = red + NW * NB;
  double* wv = par + 3 * NB;
  double* Gs = wv + NB + 2;
  double* exchG = Gs + NP;
  double* scratch = exchG + 16 * NP;
  double* slice = scratch + NQ * NP;

  const int tid = threadIdx.x, col = tid % NB, rg = tid / NB, warp = tid >> 5, lane = tid & 31;
  const long long row_lo = (long long)j0 + (long long)rank * rpc;
  long long row_hi = row_lo + rpc; if (row_hi > m) row_hi = m;
  const int nloc = row_hi > row_lo ? (int)(row_hi - row_lo) : 0;
  // pan(li, c): shared slice with pitch NB, or the matrix itself in global memory / L2
  double* const gpan = V + row_lo * ld + j0;
  const long long LD = SMEM ? NB : ld;
  double* const pan = SMEM ? slice : gpan;
  if (SMEM) {
    for (int idx = tid; idx < nloc * NB; idx += NT) {
      int li = idx / NB, c = idx % NB;
      slice[idx] = c < nbw ? gpan[(long long)li * ld + c] : 0.0;
    }
  }
  __syncthreads();
  cluster.sync();          // every CTA of the cluster is resident before the first DSMEM store

  int buf = 0;
  for (int k = 0; k < nbw; ++k) {
    const long long r = (long long)j0 + k;
    long long lo64 = r + 1 - row_lo; if (lo64 < 0) lo64 = 0; if (lo64 > nloc) lo64 = nloc;
    const int lo = (int)lo64;                                   // first local row strictly below the diagonal
    const int li0 = lo <= rg ? rg : rg + ((lo - rg + NRG - 1) / NRG) * NRG;
    const bool owner = (r >= row_lo && r < row_hi);
    double acc = 0.0;
    if (col >= k && col < nbw) {
      const double* pk = pan + (long long)li0 * LD + k;
      const double* pc = pan + (long long)li0 * LD + col;
      double a0 = 0.0, a1 = 0.0;
      int li = li0;
      for (; li + NRG < nloc; li += 2 * NRG, pk += 2 * NRG * LD, pc += 2 * NRG * LD) {
        a0 = fma(pk[0], pc[0], a0);
        a1 = fma(pk[NRG * LD], pc[NRG * LD], a1);
      }
      if (li < nloc) a0 = fma(pk[0], pc[0], a0);
      acc = a0 + a1;
    }
    if (NB == 16) acc += __shfl_xor_sync(0xffffffffu, acc, 16);
    if (lane < NB) red[warp * NB + lane] = acc;
    __syncthreads();
    if (tid < NB) {
      double g = 0.0;
#pragma unroll
      for (int w = 0; w < NW; ++w) g += red[w * NB + tid];
      double rv = owner ? pan[(r - row_lo) * LD + tid] : 0.0;
      for (int q = 0; q < C; ++q) {
        double* rex = cluster.map_shared_rank(exch, q);
        rex[(buf * 16 + rank) * NB + tid] = g;
        if (owner) { double* rr = cluster.map_shared_rank(rowv, q); rr[buf * NB + tid] = rv; }
      }
    }
    cluster.sync();
    if (tid < NB) {
      double gk = 0.0, gj = 0.0;
      for (int q = 0; q < C; ++q) { gk += exch[(buf * 16 + q) * NB + k]; gj += exch[(buf * 16 + q) * NB + tid]; }
      const double alpha = rowv[buf * NB + k], yrj = rowv[buf * NB + tid];
      double tk = 0.0, scale = 0.0, beta = alpha;
      if (gk > 0.0) {
        double sigma = sqrt(fma(alpha, alpha, gk));
        beta = alpha >= 0.0 ? -sigma : sigma;
        tk = (beta - alpha) / beta;
        scale = 1.0 / (alpha - beta);
      }
      wv[tid] = tk * fma(scale, gj, yrj);
      if (tid == 0) { par[k] = scale; par[NB + k] = beta; par[2 * NB + k] = tk; wv[NB] = scale; wv[NB + 1] = tk; }
    }
    __syncthreads();
    const double tk = wv[NB + 1];
    if (col > k && col < nbw && tk != 0.0) {
      const double w = wv[col], scale = wv[NB];
      const double* pk = pan + (long long)li0 * LD + k;
      double* pc = pan + (long long)li0 * LD + col;
      for (int li = li0; li < nloc; li += NRG, pk += NRG * LD, pc += NRG * LD)
        pc[0] = fma(-(pk[0] * scale), w, pc[0]);
      if (owner && rg == 0) pan[(r - row_lo) * LD + col] -= w;
    }
    __syncthreads();
    buf ^= 1;
  }

  // write-back: in-place factor (R above/on the diagonal, scaled v below), clean reflectors Vc
  double* const gvc = Vc + row_lo * ld + j0;
  for (int idx = tid; idx < nloc * NB; idx += NT) {
    int li = idx / NB, c = idx % NB;
    if (c >= nbw) continue;
    long long gi = row_lo + li, rc = (long long)j0 + c;
    double x = pan[(long long)li * LD + c], vout, vclean;
    if (gi > rc) { vclean = x * par[c]; vout = vclean; }
    else if (gi == rc) { vclean = 1.0; vout = par[NB + c]; }
    else { vclean = 0.0; vout = x; }
    gpan[(long long)li * ld + c] = vout;
    gvc[(long long)li * ld + c] = vclean;
    if (SMEM) slice[idx] = vclean;
  }
  if (rank == 0 && tid < nbw) tau[j0 + tid] = par[2 * NB + tid];
  __syncthreads();

  // Gram of the clean reflectors (strict upper part is what larft needs)
  {
    const int pidx = tid % NP, a = pidx / NB, c = pidx % NB, qs = tid / NP;
    const double* gsrc = SMEM ? slice : gvc;
    double g0 = 0.0, g1 = 0.0;
    if (tid < NP * NQ && a < c && c < nbw) {
      int li = qs;
      for (; li + NQ < nloc; li += 2 * NQ) {
        g0 = fma(gsrc[(long long)li * LD + a], gsrc[(long long)li * LD + c], g0);
        g1 = fma(gsrc[(long long)(li + NQ) * LD + a], gsrc[(long long)(li + NQ) * LD + c], g1);
      }
      if (li < nloc) g0 = fma(gsrc[(long long)li * LD + a], gsrc[(long long)li * LD + c], g0);
    }
    if (tid < NP * NQ) scratch[qs * NP + pidx] = g0 + g1;
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

// ------------------------------------------------------------------------------
// Register-resident panel kernel (the default).  Same algorithm as the shared-memory kernel above, but
// every thread keeps its RPT rows of its column in REGISTERS and column k is broadcast inside the
// (half-)warp with shuffles, so a column step costs no shared-memory traffic for the panel itself (the
// shared-memory version is bound by the 128 B/clk LDS bandwidth: ncu, profiles/).  All NB lanes take part
// in the dot products: lanes j >= k give the reflector/update terms g_j, lanes a < k give
// h_a = sum_{i>r} x_a[i] x_k[i], from which the Gram entries of the compact-WY recurrence follow at no
// extra pass:  G[a][k] = v_a^T v_k = scale_a (scale_k h_a + x_a[r]).  Further: (1) the diagonal row r of
// step k is taken out of the register
// tile at the START of the step (its values travel through `rowv`, its final R / v
// entries are written straight to global memory), so the register tile only ever
// holds rows strictly below the current diagonal and the dot / update loops carry no
// per-row predicates; (2) every thread finishes the reflector scalars (sqrt, two
// divisions) redundantly from the exchanged partial sums, so a column step needs ONE
// __syncthreads and (multi-CTA only) ONE cluster barrier; (3) the compact-WY column
// of T is built by warp 0 with shuffles off the critical path of the other warps.
// The panel's diagonal rows j0..j0+nbw-1 are the first local rows of rank 0 (t = 0).
// --- DSMEM exchange primitives: remote store that completes bytes on the destination CTA's mbarrier
__device__ __forceinline__ uint32_t qr_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t qr_mapa(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void qr_st_async(uint32_t remote_addr, double v, uint32_t remote_bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];\n"
               :: "r"(remote_addr), "l"(__double_as_longlong(v)), "r"(remote_bar) : "memory");
}
__device__ __forceinline__ void qr_mbar_init(uint64_t* b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" :: "r"(qr_smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void qr_mbar_arm(uint64_t* b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(qr_smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void qr_mbar_wait(uint64_t* b, uint32_t parity) {
  asm volatile(
      "{\n.reg .pred p;\nQRW_%=:\n"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
      "@p bra QRD_%=;\nbra QRW_%=;\nQRD_%=:\n}\n" :: "r"(qr_smem_u32(b)), "r"(parity) : "memory");
}
#ifndef QR_STAMP
#define QR_STAMP(i) do { } while (0)      // phase time stamps for the measurement harness (profiles/r1_qr_panel_phases.md)
#endif

// KEEPX = true: the broadcast column k (xs[]) stays in registers from the dot products to the update (RPT = 40: 640
// rows per CTA).  KEEPX = false: it is shuffled again for the update instead, which frees the registers for twice the
// rows per thread (RPT = 80: 1280 rows per CTA, 20480 per 16-CTA cluster) at ~2x the per-column time - still twice as
// fast as the shared-memory panel kernel that tall panels fell back to.
template <int NB, int NT, int RPT, bool CLUSTER, bool KEEPX = true>
__global__ void __launch_bounds__(NT, 1)
qr_panel_reg2_kernel(double* __restrict__ V, long long ld, long long m, int j0, int nbw,
                     double* __restrict__ Vc, double* __restrict__ tau, double* __restrict__ Tp, long long rpc) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int C = CLUSTER ? (int)cluster.num_blocks() : 1;
  const int rank = CLUSTER ? (int)cluster.block_rank() : 0;
  constexpr int NRG = NT / NB, NW = NT / 32;
  static_assert(NRG >= NB, "diagonal rows must all sit at t = 0");
  static_assert(RPT % 8 == 0 && NW % 4 == 0, "unrolled accumulators / tree sums");
  __shared__ double exch[2 * 16 * NB];
  __shared__ double rowv[2 * NB];
  __shared__ double red[2 * NW * NB];
  __shared__ uint64_t xbar[2];                 // per-buffer mbarrier: bytes of all ranks' partials + the diagonal row
  __shared__ double Gs[NB * NB];               // Gs[a][k] = v_a^T v_k (a < k), filled column by column
  __shared__ double taus[NB];
  __shared__ double Ts[NB * NB];

  const int tid = threadIdx.x, col = tid % NB, rg = tid / NB, warp = tid >> 5, lane = tid & 31;
  const int lane_base = lane & ~(NB - 1);
  const long long row_lo = (long long)j0 + (long long)rank * rpc;
  long long row_hi = row_lo + rpc; if (row_hi > m) row_hi = m;
  const int nloc = row_hi > row_lo ? (int)(row_hi - row_lo) : 0;
  double* const gpan = V + row_lo * ld + j0;
  double* const gvc = Vc + row_lo * ld + j0;

  double val[RPT];
  {
    const double* pl = gpan + (long long)rg * ld + col;
#pragma unroll
    for (int t = 0; t < RPT; ++t, pl += (long long)NRG * ld)
      val[t] = (rg + t * NRG < nloc && col < nbw) ? *pl : 0.0;
  }
  for (int i = tid; i < NB * NB; i += NT) { Ts[i] = 0.0; Gs[i] = 0.0; }
  if (CLUSTER && tid == 0) {
    qr_mbar_init(&xbar[0], 1); qr_mbar_init(&xbar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  double my_scale = 0.0;                       // scale of this thread's column once it has been factored
  __syncthreads();
  if (CLUSTER) cluster.sync();
  const uint32_t exch_a = qr_smem_u32(exch), rowv_a = qr_smem_u32(rowv);

  int buf = 0;
  for (int k = 0; k < nbw; ++k) {
    // A. take the diagonal row r = j0 + k out of the tile (rank 0, row group k, t = 0)
    const bool mine = (rank == 0) && (rg == k);
    double rvv = 0.0;
    if (mine) {
      rvv = val[0]; val[0] = 0.0;
      if (CLUSTER) {
        for (int q = 0; q < C; ++q)
          qr_st_async(qr_mapa(rowv_a + (buf * NB + col) * 8, q), rvv, qr_mapa(qr_smem_u32(&xbar[buf]), q));
      } else rowv[buf * NB + col] = rvv;
    }
    // B. column k of my rows, dot with my column.  FP64 dependent-issue latency is long (~30 cycles),
    //    so the sum runs on 8 independent accumulators combined by a fixed tree.
    double xs[KEEPX ? RPT : 1];
    double ac[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) ac[u] = 0.0;
#pragma unroll
    for (int t = 0; t < RPT; ++t) {
      const double x = __shfl_sync(0xffffffffu, val[t], lane_base | k);
      if (KEEPX) xs[t] = x;
      ac[t & 7] = fma(x, val[t], ac[t & 7]);
    }
    double acc = ((ac[0] + ac[1]) + (ac[2] + ac[3])) + ((ac[4] + ac[5]) + (ac[6] + ac[7]));
    if (NB == 16) acc += __shfl_xor_sync(0xffffffffu, acc, 16);
    if (lane < NB) red[(buf * NW + warp) * NB + lane] = acc;
    __syncthreads();
    double gk = 0.0, gj = 0.0;
    if (CLUSTER) {
      // every thread sums the warps' partials of ITS column (fixed tree), thread (q = tid / NB) sends it to rank q
      if (tid == 0) qr_mbar_arm(&xbar[buf], (uint32_t)(C * NB + NB) * 8u);
      {
        double pg[NW];
#pragma unroll
        for (int w = 0; w < NW; ++w) pg[w] = red[(buf * NW + w) * NB + col];
#pragma unroll
        for (int st = 1; st < NW; st *= 2)
#pragma unroll
          for (int w = 0; w + st < NW; w += 2 * st) pg[w] += pg[w + st];
        for (int q = rg; q < C; q += NRG)
          qr_st_async(qr_mapa(exch_a + ((buf * 16 + rank) * NB + col) * 8, q), pg[0], qr_mapa(qr_smem_u32(&xbar[buf]), q));
      }
      qr_mbar_wait(&xbar[buf], (k >> 1) & 1);
      double pk[16], pj[16];
#pragma unroll
      for (int q = 0; q < 16; ++q) {
        pk[q] = q < C ? exch[(buf * 16 + q) * NB + k] : 0.0;
        pj[q] = q < C ? exch[(buf * 16 + q) * NB + col] : 0.0;
      }
#pragma unroll
      for (int st = 1; st < 16; st *= 2)
#pragma unroll
        for (int q = 0; q + st < 16; q += 2 * st) { pk[q] += pk[q + st]; pj[q] += pj[q + st]; }
      gk = pk[0]; gj = pj[0];
    } else {
      double pk[NW], pj[NW];
#pragma unroll
      for (int w = 0; w < NW; ++w) { pk[w] = red[(buf * NW + w) * NB + k]; pj[w] = red[(buf * NW + w) * NB + col]; }
#pragma unroll
      for (int st = 1; st < NW; st *= 2)
#pragma unroll
        for (int w = 0; w + st < NW; w += 2 * st) { pk[w] += pk[w + st]; pj[w] += pj[w + st]; }
      gk = pk[0]; gj = pj[0];
    }
    // F. reflector scalars (identical in every thread)
    const double alpha = rowv[buf * NB + k], yrj = rowv[buf * NB + col];
    double tk = 0.0, scale = 0.0, beta = alpha;
    if (gk > 0.0) {
      const double sigma = sqrt(fma(alpha, alpha, gk));
      beta = alpha >= 0.0 ? -sigma : sigma;
      tk = (beta - alpha) / beta;
      scale = 1.0 / (alpha - beta);
    }
    const double z = fma(scale, gj, yrj);          // v_k^T y_j (j > k)  or  (x_a[r] + scale h_a) (a < k)
    const double w = tk * z;
    // G. update the trailing panel columns
    if (KEEPX) {
      if (col > k && col < nbw && tk != 0.0) {
        const double nsw = -scale * w;
#pragma unroll
        for (int t = 0; t < RPT; ++t) val[t] = fma(xs[t], nsw, val[t]);
      }
    } else {
      // all lanes take part in the shuffles; column k itself (nsw = 0 there) is not modified, so the values read are
      // the ones the dot products saw
      const double nsw = (col > k && col < nbw && tk != 0.0) ? -scale * w : 0.0;
#pragma unroll
      for (int t = 0; t < RPT; ++t) {
        const double x = __shfl_sync(0xffffffffu, val[t], lane_base | k);
        if (nsw != 0.0) val[t] = fma(x, nsw, val[t]);
      }
    }
    // H. final entries of row r
    if (mine && col < nbw) {
      double vout, vclean;
      if (col < k) { vclean = rvv * my_scale; vout = vclean; }
      else if (col == k) { vclean = 1.0; vout = beta; }
      else { vclean = 0.0; vout = (tk != 0.0) ? rvv - w : rvv; }
      V[(long long)(j0 + k) * ld + j0 + col] = vout;
      Vc[(long long)(j0 + k) * ld + j0 + col] = vclean;
    }
    // I. Gram column k of the reflectors (for the T factor, built after the loop) and tau_k
    if (rg == 0) {
      if (col < k) Gs[col * NB + k] = my_scale * z;
      else if (col == k) { taus[k] = tk; if (rank == 0) tau[j0 + k] = tk; }
    }
    if (col == k) my_scale = scale;
    buf ^= 1;
  }

  // write-back of the rows below the panel's diagonal block
  if (col < nbw) {
    double* po = gpan + (long long)rg * ld + col;
    double* pc = gvc + (long long)rg * ld + col;
#pragma unroll
    for (int t = 0; t < RPT; ++t, po += (long long)NRG * ld, pc += (long long)NRG * ld) {
      const int li = rg + t * NRG;
      if (li < nloc && !(rank == 0 && li < nbw)) {
        const double v = val[t] * my_scale;
        *po = v; *pc = v;
      }
    }
  }
  // compact-WY factor, forward recurrence (LAPACK dlarft): T[a][k] = -tau_k sum_{c=a}^{k-1} T[a][c] G[c][k]
  __syncthreads();
  if (rank == 0 && warp == 0) {
    if (lane < NB) {
      const int a = lane;
      for (int k = 0; k < nbw; ++k) {
        const double tk = taus[k];
        if (a == k) Ts[k * NB + k] = tk;
        else if (a < k) {
          double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
          for (int c = 0; c < NB; c += 4) {
            if (c >= a && c < k) s0 = fma(Ts[a * NB + c], Gs[c * NB + k], s0);
            if (c + 1 >= a && c + 1 < k) s1 = fma(Ts[a * NB + c + 1], Gs[(c + 1) * NB + k], s1);
            if (c + 2 >= a && c + 2 < k) s2 = fma(Ts[a * NB + c + 2], Gs[(c + 2) * NB + k], s2);
            if (c + 3 >= a && c + 3 < k) s3 = fma(Ts[a * NB + c + 3], Gs[(c + 3) * NB + k], s3);
          }
          Ts[a * NB + k] = -tk * ((s0 + s1) + (s2 + s3));
        }
      }
    }
    __syncwarp();
    for (int i = lane; i < NB * NB; i += 32) Tp[i] = Ts[i];
  }
  if (CLUSTER) cluster.sync();      // nobody exits while a peer may still address its shared memory
}

// ------------------------------------------------------------------------------
// Whole-matrix register-resident QR (small / medium c~: n <= 16 NCS columns, rows <= 16 RPT per CTA, up to 16 CTAs).
// Same column step as qr_panel_reg2_kernel, but every thread holds its rows of ALL its NCS column slots
// (column c = cs*16 + tid%16), so the Householder update of the whole trailing matrix happens in registers:
// no panel / WY-apply launches at all.  The dots of column k with every other column come out of one reduction:
// columns j > k feed the update, columns a < k give the Gram entries G[a][k] = v_a^T v_k, i.e. the complete
// V^T V that the one-shot form-Q (wy_formq_trsm_kernel) needs, plus the per-block T_p.  Outputs: R (upper
// triangle, rows written as they retire), the clean reflectors Vc, tau, G (n x n) and the T_p blocks.
template <int NCS, int RPT, bool CLUSTER>
__global__ void __launch_bounds__(256, 1)
qr_full_reg_kernel(const double* __restrict__ X, long long ld, long long m, int n, double* __restrict__ Rout,
                   double* __restrict__ Vc, double* __restrict__ tau, double* __restrict__ Gout,
                   double* __restrict__ Tfac, long long rpc) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int C = CLUSTER ? (int)cluster.num_blocks() : 1;
  const int rank = CLUSTER ? (int)cluster.block_rank() : 0;
  constexpr int NB = 16, NT = 256, NRG = NT / NB, NW = NT / 32, NP = NCS * NB;   // NP: padded column count
  static_assert(RPT >= NCS, "the diagonal rows of column slot cs sit at t = cs");
  extern __shared__ __align__(16) double fsm[];
  double* exch = fsm;                       // [2][16][NP]
  double* rowv = exch + 2 * 16 * NP;        // [2][NP]
  double* red = rowv + 2 * NP;              // [2][NW][NP]
  double* gsum = red + 2 * NW * NP;         // [NP]   cluster-wide sums of the current column step
  double* Gs = gsum + NP;                   // [NP][NP]
  double* taus = Gs + NP * NP;              // [NP]
  double* scl = taus + NP;                  // [NP]   scale of every factored column
  __shared__ uint64_t xbar[2];

  const int tid = threadIdx.x, col = tid % NB, rg = tid / NB, warp = tid >> 5, lane = tid & 31;
  const int lane_base = lane & ~(NB - 1);
  const long long row_lo = (long long)rank * rpc;
  long long row_hi = row_lo + rpc; if (row_hi > m) row_hi = m;
  const int nloc = row_hi > row_lo ? (int)(row_hi - row_lo) : 0;

  double val[NCS][RPT];
#pragma unroll
  for (int cs = 0; cs < NCS; ++cs)
#pragma unroll
    for (int t = 0; t < RPT; ++t) {
      const int li = rg + t * NRG, c = cs * NB + col;
      val[cs][t] = (li < nloc && c < n) ? X[(row_lo + li) * ld + c] : 0.0;
    }
  for (int i = tid; i < NP * NP; i += NT) Gs[i] = 0.0;
  for (int i = tid; i < NP; i += NT) { taus[i] = 0.0; scl[i] = 0.0; }
  if (CLUSTER && tid == 0) {
    qr_mbar_init(&xbar[0], 1); qr_mbar_init(&xbar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  if (CLUSTER) cluster.sync();
  const uint32_t exch_a = qr_smem_u32(exch), rowv_a = qr_smem_u32(rowv);

  int buf = 0, kidx = 0;
#pragma unroll
  for (int csk = 0; csk < NCS; ++csk) {
    for (int kk = 0; kk < NB; ++kk, ++kidx) {
      const int k = csk * NB + kk;
      if (k >= n) break;
      // A. retire the diagonal row r = k: rank 0, row group kk, t = csk (static)
      const bool mine = (rank == 0) && (rg == kk);
      double rvv[NCS];
#pragma unroll
      for (int cs = 0; cs < NCS; ++cs) rvv[cs] = 0.0;
      if (mine) {
#pragma unroll
        for (int cs = 0; cs < NCS; ++cs) {
          rvv[cs] = val[cs][csk]; val[cs][csk] = 0.0;
          if (CLUSTER) {
            for (int q = 0; q < C; ++q)
              qr_st_async(qr_mapa(rowv_a + (buf * NP + cs * NB + col) * 8, q), rvv[cs], qr_mapa(qr_smem_u32(&xbar[buf]), q));
          } else rowv[buf * NP + cs * NB + col] = rvv[cs];
        }
      }
      // B. column k of my rows (shuffle broadcast inside the half warp), dots with all my columns
      double xs[RPT], acc[NCS];
#pragma unroll
      for (int cs = 0; cs < NCS; ++cs) acc[cs] = 0.0;
#pragma unroll
      for (int t = 0; t < RPT; ++t) {
        xs[t] = __shfl_sync(0xffffffffu, val[csk][t], lane_base | kk);
#pragma unroll
        for (int cs = 0; cs < NCS; ++cs) acc[cs] = fma(xs[t], val[cs][t], acc[cs]);
      }
#pragma unroll
      for (int cs = 0; cs < NCS; ++cs) {
        acc[cs] += __shfl_xor_sync(0xffffffffu, acc[cs], 16);
        if (lane < NB) red[(buf * NW + warp) * NP + cs * NB + lane] = acc[cs];
      }
      __syncthreads();
      // C. CTA sums (fixed tree over the warps), then the cluster exchange
      if (CLUSTER) {
        if (tid == 0) qr_mbar_arm(&xbar[buf], (uint32_t)(C * NP + NP) * 8u);
        for (int e = tid; e < NP * 16; e += NT) {              // (destination rank q, column c)
          const int c = e % NP, q = e / NP;
          if (q < C) {
            double pg[NW];
#pragma unroll
            for (int w = 0; w < NW; ++w) pg[w] = red[(buf * NW + w) * NP + c];
#pragma unroll
            for (int st = 1; st < NW; st *= 2)
#pragma unroll
              for (int w = 0; w + st < NW; w += 2 * st) pg[w] += pg[w + st];
            qr_st_async(qr_mapa(exch_a + ((buf * 16 + rank) * NP + c) * 8, q), pg[0], qr_mapa(qr_smem_u32(&xbar[buf]), q));
          }
        }
        qr_mbar_wait(&xbar[buf], (kidx >> 1) & 1);
        if (tid < NP) {
          double pk[16];
#pragma unroll
          for (int q = 0; q < 16; ++q) pk[q] = q < C ? exch[(buf * 16 + q) * NP + tid] : 0.0;
#pragma unroll
          for (int st = 1; st < 16; st *= 2)
#pragma unroll
            for (int q = 0; q + st < 16; q += 2 * st) pk[q] += pk[q + st];
          gsum[tid] = pk[0];
        }
      } else {
        if (tid < NP) {
          double pg[NW];
#pragma unroll
          for (int w = 0; w < NW; ++w) pg[w] = red[(buf * NW + w) * NP + tid];
#pragma unroll
          for (int st = 1; st < NW; st *= 2)
#pragma unroll
            for (int w = 0; w + st < NW; w += 2 * st) pg[w] += pg[w + st];
          gsum[tid] = pg[0];
        }
      }
      __syncthreads();
      // F. reflector scalars (identical in every thread)
      const double gk = gsum[k], alpha = rowv[buf * NP + k];
      double tk = 0.0, scale = 0.0, beta = alpha;
      if (gk > 0.0) {
        const double sigma = sqrt(fma(alpha, alpha, gk));
        beta = alpha >= 0.0 ? -sigma : sigma;
        tk = (beta - alpha) / beta;
        scale = 1.0 / (alpha - beta);
      }
      // G/H/I. per column slot: update (columns > k), final row-r entries, Gram column (columns < k)
#pragma unroll
      for (int cs = 0; cs < NCS; ++cs) {
        const int c = cs * NB + col;
        const double z = fma(scale, gsum[c], rowv[buf * NP + c]);
        const double w = tk * z;
        if (c > k && c < n && tk != 0.0) {
          const double nsw = -scale * w;
#pragma unroll
          for (int t = 0; t < RPT; ++t) val[cs][t] = fma(xs[t], nsw, val[cs][t]);
        }
        if (mine && c < n) {
          const double sc_c = scl[c];
          double vclean, rval;
          if (c < k) { vclean = rvv[cs] * sc_c; rval = 0.0; }
          else if (c == k) { vclean = 1.0; rval = beta; }
          else { vclean = 0.0; rval = (tk != 0.0) ? rvv[cs] - w : rvv[cs]; }
          Vc[(long long)k * ld + c] = vclean;
          Rout[(long long)k * n + c] = rval;
        }
        if (rg == 0 && c < k) Gs[c * NP + k] = scl[c] * z;
      }
      __syncthreads();                                   // everyone has read scl / gsum / rowv of this step
      if (tid == 0) { taus[k] = tk; scl[k] = scale; if (rank == 0) tau[k] = tk; }
      buf ^= 1;
    }
  }
  __syncthreads();

  // clean reflectors below the diagonal rows
#pragma unroll
  for (int cs = 0; cs < NCS; ++cs) {
    const int c = cs * NB + col;
    if (c < n) {
      const double sc_c = scl[c];
#pragma unroll
      for (int t = 0; t < RPT; ++t) {
        const int li = rg + t * NRG;
        const long long gi = row_lo + li;
        if (li < nloc && gi >= n) Vc[gi * ld + c] = val[cs][t] * sc_c;     // rows < n were written when they retired
      }
    }
  }
  if (rank == 0) {
    // G (strict upper part is what the solve needs) and the per-block compact-WY factors T_p
    for (int i = tid; i < n * n; i += NT) { const int a = i / n, c = i % n; Gout[i] = Gs[a * NP + c]; }
    if (warp == 0 && lane < NB) {
      const int a = lane;
      for (int p = 0; p * NB < n; ++p) {
        double Trow[NB];
#pragma unroll
        for (int i = 0; i < NB; ++i) Trow[i] = 0.0;
#pragma unroll
        for (int i = 0; i < NB; ++i) {
          const int gi = p * NB + i;
          if (gi < n) {
            const double ti = taus[gi];
            if (a == i) Trow[i] = ti;
            else if (a < i) {
              double sacc = 0.0;
#pragma unroll
              for (int c = 0; c < NB; ++c)
                if (c >= a && c < i) sacc = fma(Trow[c], Gs[(p * NB + c) * NP + gi], sacc);
              Trow[i] = -ti * sacc;
            }
          }
        }
#pragma unroll
        for (int i = 0; i < NB; ++i) Tfac[(size_t)p * NB * NB + a * NB + i] = Trow[i];
      }
    }
  }
  if (CLUSTER) cluster.sync();
}

// ------------------------------------------------------------------------------
// Applying a block reflector  Y <- (I - Vp op(T) Vp^T) Y  to Y = rows x nc (ld ldy):
// three memory-bound kernels (intensity 2*NB flop per 16 bytes of Y, below the
// FP64 ridge of ~5.7 flop/B even at NB = 32, so plain DFMA with coalesced row
// streaming, not tensor tiles):
//   wy_partial : part[cta][a][j] = sum_{i in chunk} Vp[i][a] Y[i][j]
//   wy_reduce  : W2[a][j] = sum_k opT(a,k) sum_cta part[cta][k][j]      (fixed order)
//   wy_update  : Y[i][j] -= sum_a Vp[i][a] W2[a][j]
// One thread per column j (nc <= 4 * blockDim).
template <int NB>
__global__ void __launch_bounds__(256)
wy_partial_kernel(const double* __restrict__ Vp, long long ldv, const double* __restrict__ Y, long long ldy,
                  long long rows, int nc, int nbw, int chunk, double* __restrict__ part) {
  __shared__ double vs[64 * NB];
  const long long r0 = (long long)blockIdx.x * chunk;
  long long r1 = r0 + chunk; if (r1 > rows) r1 = rows;
  const int tid = threadIdx.x;
  for (int j0c = 0; j0c < nc; j0c += 256) {
    const int j = j0c + tid;
    double acc[NB];
#pragma unroll
    for (int a = 0; a < NB; ++a) acc[a] = 0.0;
    for (long long rb = r0; rb < r1; rb += 64) {
      const int nr = (int)((r1 - rb) < 64 ? (r1 - rb) : 64);
      __syncthreads();
      for (int idx = tid; idx < nr * NB; idx += 256) {
        int i = idx / NB, a = idx % NB;
        vs[idx] = a < nbw ? Vp[(rb + i) * ldv + a] : 0.0;
      }
      __syncthreads();
      if (j < nc) {
        int i = 0;
        for (; i + 4 <= nr; i += 4) {
          double y0 = Y[(rb + i) * ldy + j], y1 = Y[(rb + i + 1) * ldy + j], y2 = Y[(rb + i + 2) * ldy + j],
                 y3 = Y[(rb + i + 3) * ldy + j];
#pragma unroll
          for (int a = 0; a < NB; ++a) {
            acc[a] = fma(vs[i * NB + a], y0, acc[a]);
            acc[a] = fma(vs[(i + 1) * NB + a], y1, acc[a]);
            acc[a] = fma(vs[(i + 2) * NB + a], y2, acc[a]);
            acc[a] = fma(vs[(i + 3) * NB + a], y3, acc[a]);
          }
        }
        for (; i < nr; ++i) {
          double y0 = Y[(rb + i) * ldy + j];
#pragma unroll
          for (int a = 0; a < NB; ++a) acc[a] = fma(vs[i * NB + a], y0, acc[a]);
        }
      }
    }
    if (j < nc) {
#pragma unroll
      for (int a = 0; a < NB; ++a) part[((long long)blockIdx.x * NB + a) * nc + j] = acc[a];
    }
  }
}

// grid: ceil(nc / 4) blocks; block = 4 columns x NB rows k (= 4*NB elements) x NG part-groups.
// Thread (e, g) sums the parts c == g (mod NG) of element e with coalesced loads, the NG
// group sums are added in fixed order, then W2 = op(T) W1 for the block's 4 columns.
template <int NB>
__global__ void __launch_bounds__(1024)
wy_reduce_kernel(const double* __restrict__ part, int nparts, int nc, int nbw, const double* __restrict__ Tp,
                 int transT, double* __restrict__ W2) {
  constexpr int NE = 4 * NB, NG = 1024 / NE;
  __shared__ double gs[NG * NE];
  __shared__ double w1[NE];
  const int e = threadIdx.x % NE, g = threadIdx.x / NE;
  const int k = e / 4, jj = e % 4, j = blockIdx.x * 4 + jj;
  double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
  if (j < nc && k < nbw) {
    const double* p = part + (long long)k * nc + j;
    const long long st = (long long)NB * nc;
    int c = g;
    for (; c + 3 * NG < nparts; c += 4 * NG) {
      double v0 = p[(long long)c * st], v1 = p[(long long)(c + NG) * st], v2 = p[(long long)(c + 2 * NG) * st],
             v3 = p[(long long)(c + 3 * NG) * st];
      s0 += v0; s1 += v1; s2 += v2; s3 += v3;
    }
    for (; c < nparts; c += NG) s0 += p[(long long)c * st];
  }
  gs[g * NE + e] = (s0 + s1) + (s2 + s3);
  __syncthreads();
  if (threadIdx.x < NE) {
    double t = 0.0;
#pragma unroll
    for (int q = 0; q < NG; ++q) t += gs[q * NE + threadIdx.x];
    w1[threadIdx.x] = t;
  }
  __syncthreads();
  if (threadIdx.x < NE) {
    const int a = k;                 // reuse the (k, jj) decomposition as (a, jj)
    if (j < nc && a < nbw) {
      double s = 0.0;
      for (int kk = 0; kk < nbw; ++kk) {
        const double t = transT ? Tp[kk * NB + a] : Tp[a * NB + kk];
        s = fma(t, w1[kk * 4 + jj], s);
      }
      W2[(long long)a * nc + j] = s;
    }
  }
}

template <int NB>
__global__ void __launch_bounds__(256)
wy_update_kernel(const double* __restrict__ Vp, long long ldv, double* __restrict__ Y, long long ldy,
                 long long rows, int nc, int nbw, int chunk, const double* __restrict__ W2) {
  __shared__ double vs[64 * NB];
  const long long r0 = (long long)blockIdx.x * chunk;
  long long r1 = r0 + chunk; if (r1 > rows) r1 = rows;
  const int tid = threadIdx.x;
  for (int j0c = 0; j0c < nc; j0c += 256) {
    const int j = j0c + tid;
    double w[NB];
#pragma unroll
    for (int a = 0; a < NB; ++a) w[a] = (j < nc && a < nbw) ? W2[(long long)a * nc + j] : 0.0;
    for (long long rb = r0; rb < r1; rb += 64) {
      const int nr = (int)((r1 - rb) < 64 ? (r1 - rb) : 64);
      __syncthreads();
      for (int idx = tid; idx < nr * NB; idx += 256) {
        int i = idx / NB, a = idx % NB;
        vs[idx] = a < nbw ? Vp[(rb + i) * ldv + a] : 0.0;
      }
      __syncthreads();
      if (j < nc) {
        int i = 0;
        for (; i + 4 <= nr; i += 4) {
          double* y = Y + (rb + i) * ldy + j;
          double y0 = y[0], y1 = y[ldy], y2 = y[2 * ldy], y3 = y[3 * ldy];
          double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
          for (int a = 0; a < NB; ++a) {
            s0 = fma(vs[i * NB + a], w[a], s0);
            s1 = fma(vs[(i + 1) * NB + a], w[a], s1);
            s2 = fma(vs[(i + 2) * NB + a], w[a], s2);
            s3 = fma(vs[(i + 3) * NB + a], w[a], s3);
          }
          y[0] = y0 - s0; y[ldy] = y1 - s1; y[2 * ldy] = y2 - s2; y[3 * ldy] = y3 - s3;
        }
        for (; i < nr; ++i) {
          double* y = Y + (rb + i) * ldy + j;
          double s0 = 0.0;
#pragma unroll
          for (int a = 0; a < NB; ++a) s0 = fma(vs[i * NB + a], w[a], s0);
          y[0] -= s0;
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------
// The same block-reflector application in ONE launch (trailing update of the blocked QR):
//   Y <- (I - Vp op(T) Vp^T) Y,   Y = rows x nc (ld ldy),  Vp = rows x nbw (ld ldv)
// A cluster of CS CTAs owns a slab of 16 columns of Y and all its rows (CTA rank r: a contiguous block of
// rows_cta rows).  Each thread keeps its part of the slab in registers from the one read to the one write
// (2 columns x RPT rows; thread = (row group rg = tid / 8, column pair ct = tid % 8), rows rg + 32 i); the CTA's
// rows of Vp sit in shared memory (pitch 18 doubles: the four rows a warp touches fall into different banks).
//   phase 1: W1 = Vp^T Y     per-thread partial sums -> warp shuffles -> 8 warps (fixed order) -> the cluster's
//                            CTAs through distributed shared memory (fixed order over the ranks)
//   phase 2: W2 = op(T) W1   16 x 16, every CTA for itself
//   phase 3: Y -= Vp W2      from the registers, one coalesced write
// Y crosses the L2 once in each direction (the three-kernel version reads it twice and goes through `part`), and the
// two relaunches are gone.  Deterministic: every sum has a fixed order.
template <int NB, int RPT>
__global__ void __launch_bounds__(256, 1)
wy_fused_cluster_kernel(const double* __restrict__ Vp, long long ldv, double* __restrict__ Y, long long ldy,
                        long long rows, int nc, int nbw, const double* __restrict__ Tp, int transT, int rows_cta) {
  static_assert(NB == 16, "thread mapping assumes 16-column slabs and 16-wide panels");
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int CS = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  constexpr int VP = NB + 2;                      // shared-memory pitch of a row of Vp
  extern __shared__ __align__(16) double wsm[];
  double* vs = wsm;                               // rows_cta x VP
  double* red = vs + (size_t)rows_cta * VP;       // 8 warps x 256
  double* xch = red + 8 * 256;                    // CS ranks x 256   (written by the peers)
  double* w2s = xch + 16 * 256;                   // 16 x 16
  const int tid = threadIdx.x, rg = tid >> 3, ct = tid & 7, lane = tid & 31, warp = tid >> 5;
  const int slab = blockIdx.x / CS;
  const int jc = slab * NB + ct;                  // this thread's columns: jc, jc + 8
  const bool c0ok = jc < nc, c1ok = jc + 8 < nc;
  const long long r0 = (long long)rank * rows_cta;
  long long rl = rows - r0; if (rl > rows_cta) rl = rows_cta; if (rl < 0) rl = 0;
  const int nr = (int)rl;                         // rows of this CTA

  // the slab into registers (all loads in flight at once), the rows of Vp into shared memory
  double y0[RPT], y1[RPT];
#pragma unroll
  for (int i = 0; i < RPT; ++i) {
    const int r = rg + 32 * i;
    const double* yp = Y + (r0 + r) * ldy + jc;
    y0[i] = (r < nr && c0ok) ? yp[0] : 0.0;
    y1[i] = (r < nr && c1ok) ? yp[8] : 0.0;
  }
  {
    const int a = tid & 15;                         // 16 rows per sweep of the CTA, 8 sweeps in flight
    const double* vp = Vp + r0 * ldv + a;
    for (int ib = tid >> 4; ib < nr; ib += 128) {
      double t[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) t[u] = (a < nbw && ib + 16 * u < nr) ? vp[(long long)(ib + 16 * u) * ldv] : 0.0;
#pragma unroll
      for (int u = 0; u < 8; ++u) if (ib + 16 * u < nr) vs[(ib + 16 * u) * VP + a] = t[u];
    }
  }
  __syncthreads();

  // phase 1
  double acc0[NB], acc1[NB];
#pragma unroll
  for (int a = 0; a < NB; ++a) acc0[a] = acc1[a] = 0.0;
#pragma unroll
  for (int i = 0; i < RPT; ++i) {
    const int r = rg + 32 * i;
    if (r < nr) {
      const double2* v2 = reinterpret_cast<const double2*>(vs + r * VP);
#pragma unroll
      for (int q = 0; q < NB / 2; ++q) {
        const double2 v = v2[q];
        acc0[2 * q] = fma(v.x, y0[i], acc0[2 * q]);         acc1[2 * q] = fma(v.x, y1[i], acc1[2 * q]);
        acc0[2 * q + 1] = fma(v.y, y0[i], acc0[2 * q + 1]); acc1[2 * q + 1] = fma(v.y, y1[i], acc1[2 * q + 1]);
      }
    }
  }
  // the four row groups of a warp (lanes ct, ct+8, ct+16, ct+24), then the 8 warps in order
#pragma unroll
  for (int a = 0; a < NB; ++a) {
    acc0[a] += __shfl_xor_sync(0xffffffffu, acc0[a], 8);  acc1[a] += __shfl_xor_sync(0xffffffffu, acc1[a], 8);
    acc0[a] += __shfl_xor_sync(0xffffffffu, acc0[a], 16); acc1[a] += __shfl_xor_sync(0xffffffffu, acc1[a], 16);
  }
  if (lane < 8) {
#pragma unroll
    for (int a = 0; a < NB; ++a) {
      red[warp * 256 + a * NB + ct] = acc0[a];
      red[warp * 256 + a * NB + ct + 8] = acc1[a];
    }
  }
  __syncthreads();
  {
    double t = 0.0;                                // thread tid = entry (a, j) = (tid / 16, tid % 16)
#pragma unroll
    for (int w = 0; w < 8; ++w) t += red[w * 256 + tid];
    for (int q = 0; q < CS; ++q) *cluster.map_shared_rank(xch + rank * 256 + tid, q) = t;
  }
  cluster.sync();
  {
    double t = 0.0;
    for (int q = 0; q < CS; ++q) t += xch[q * 256 + tid];
    red[tid] = t;                                  // W1[a][j]
  }
  __syncthreads();

  // phase 2
  {
    const int a = tid >> 4, j = tid & 15;
    double t = 0.0;
    if (a < nbw)
      for (int k = 0; k < nbw; ++k) t = fma(transT ? Tp[k * NB + a] : Tp[a * NB + k], red[k * NB + j], t);
    w2s[tid] = t;
  }
  __syncthreads();

  // phase 3
  double w0[NB], w1[NB];
#pragma unroll
  for (int a = 0; a < NB; ++a) { w0[a] = w2s[a * NB + ct]; w1[a] = w2s[a * NB + ct + 8]; }
#pragma unroll
  for (int i = 0; i < RPT; ++i) {
    const int r = rg + 32 * i;
    if (r < nr) {
      const double2* v2 = reinterpret_cast<const double2*>(vs + r * VP);
      double s0 = 0.0, s1 = 0.0, t0 = 0.0, t1 = 0.0;
#pragma unroll
      for (int q = 0; q < NB / 2; ++q) {
        const double2 v = v2[q];
        s0 = fma(v.x, w0[2 * q], s0);     s1 = fma(v.x, w1[2 * q], s1);
        t0 = fma(v.y, w0[2 * q + 1], t0); t1 = fma(v.y, w1[2 * q + 1], t1);
      }
      double* yp = Y + (r0 + r) * ldy + jc;
      if (c0ok) yp[0] = y0[i] - (s0 + t0);
      if (c1ok) yp[8] = y1[i] - (s1 + t1);
    }
  }
}

// ------------------------------------------------------------------------------
// Form Q in one shot (K2c).  With all reflectors V (unit lower trapezoidal, m x n) the product of the
// Householder transformations is  H_1 ... H_n = I - V T V^T,  T^{-1} = D^{-1} + striu(V^T V), D = diag(tau),
// so  Q = (I - V T V^T) [I;0] = [I;0] - V X,   X = T V_top^T   (V_top = the first n rows of V),
// i.e. X solves the upper-triangular system (D^{-1} + striu(G)) X = V_top^T with G = V^T V.  The diagonal blocks
// of that system are inverted already: (D_p^{-1} + striu(G_pp))^{-1} = T_p, the per-panel compact-WY factors.
// Blocked back substitution, one CTA per 16 right-hand-side columns:  X_p = T_p (Y_p - sum_{q>p} G_pq X_q).
template <int NB>
__global__ void __launch_bounds__(NB * NB)
wy_formq_trsm_kernel(const double* __restrict__ G, const double* __restrict__ Tfac, const double* __restrict__ Vc,
                     long long ldv, int n, double* __restrict__ X) {
  extern __shared__ double xs_[];              // X chunk: n x NB
  __shared__ double rblk[NB * NB];
  const int a = threadIdx.x / NB, jj = threadIdx.x % NB;   // entry (a, jj) of a 16 x 16 block
  const int j = blockIdx.x * NB + jj;                       // right-hand-side column
  const int npan = (n + NB - 1) / NB;
  double* gs = xs_ + (size_t)npan * NB * NB;                // G row block: NB x (npan * NB)
  const int ldg = npan * NB;
  for (int p = npan - 1; p >= 0; --p) {
    const int ra = p * NB + a;                              // row of the system
    // stage rows p*NB .. p*NB+NB-1 of G, columns (p+1)*NB .. n-1, coalesced
    for (int idx = threadIdx.x; idx < NB * ldg; idx += NB * NB) {
      const int rr = idx / ldg, cc = idx % ldg;
      const int gr = p * NB + rr;
      gs[idx] = (gr < n && cc < n && cc >= (p + 1) * NB) ? G[(long long)gr * n + cc] : 0.0;
    }
    __syncthreads();
    double r = 0.0;
    if (ra < n && j < n) {
      r = (j >= ra) ? Vc[(long long)j * ldv + ra] : 0.0;    // Y[ra][j] = V[j][ra] (zero above the diagonal of V)
      double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
      const int c_lo = (p + 1) * NB, c_hi = npan * NB;      // padded columns hold zeros in gs and xs_
      for (int c = c_lo; c < c_hi; c += 4) {
        s0 = fma(gs[a * ldg + c], xs_[c * NB + jj], s0);
        s1 = fma(gs[a * ldg + c + 1], xs_[(c + 1) * NB + jj], s1);
        s2 = fma(gs[a * ldg + c + 2], xs_[(c + 2) * NB + jj], s2);
        s3 = fma(gs[a * ldg + c + 3], xs_[(c + 3) * NB + jj], s3);
      }
      r -= (s0 + s1) + (s2 + s3);
    }
    rblk[a * NB + jj] = r;
    __syncthreads();
    double x = 0.0;
    const double* Tp = Tfac + (size_t)p * NB * NB;
    if (ra < n) {
#pragma unroll
      for (int c = 0; c < NB; ++c) x = fma(Tp[a * NB + c], rblk[c * NB + jj], x);   // T_p upper triangular (zeros below)
      if (j < n) X[(long long)ra * n + j] = x;
    }
    xs_[ra * NB + jj] = x;                                  // padded rows: zero
    __syncthreads();
  }
}

// The same back substitution for n <= 256 with the global loads taken off the dependent chain: all T_p are staged
// once, and the G row block and right-hand-side entries of step p-1 are fetched into registers while step p is
// computed from shared memory (one global latency per kernel instead of three per block step: 62 -> ~15 us at n = 196).
template <int NB>
__global__ void __launch_bounds__(NB * NB)
wy_formq_trsm_pipe_kernel(const double* __restrict__ G, const double* __restrict__ Tfac, const double* __restrict__ Vc,
                          long long ldv, int n, double* __restrict__ X) {
  constexpr int NT = NB * NB, MAXL = 16;                    // ldg <= MAXL * NB
  extern __shared__ double xs_[];                           // X chunk: (npan * NB) x NB
  __shared__ double rblk[NT];
  const int a = threadIdx.x / NB, jj = threadIdx.x % NB;
  const int j = blockIdx.x * NB + jj;
  const int npan = (n + NB - 1) / NB, ldg = npan * NB;
  double* gs = xs_ + (size_t)ldg * NB;                      // G row block: NB x ldg
  double* ts = gs + (size_t)NB * ldg;                       // all T_p: npan x NB x NB
  for (int idx = threadIdx.x; idx < npan * NT; idx += NT) ts[idx] = Tfac[idx];
  for (int idx = threadIdx.x; idx < ldg * NB; idx += NT) xs_[idx] = 0.0;
  // prefetch registers: thread t holds elements t, t + NT, ... of the NB x ldg row block (row rr = idx / ldg)
  double gpre[MAXL], rpre;
  auto fetch = [&](int p) {
#pragma unroll
    for (int u = 0; u < MAXL; ++u) {
      const int idx = threadIdx.x + u * NT;
      const int rr = idx / ldg, cc = idx % ldg, gr = p * NB + rr;
      gpre[u] = (idx < NB * ldg && gr < n && cc < n && cc >= (p + 1) * NB) ? G[(long long)gr * n + cc] : 0.0;
    }
    const int ra = p * NB + a;
    rpre = (ra < n && j < n && j >= ra) ? Vc[(long long)j * ldv + ra] : 0.0;   // Y[ra][j] = V[j][ra]
  };
  fetch(npan - 1);
  for (int p = npan - 1; p >= 0; --p) {
    const int ra = p * NB + a;
    __syncthreads();                                        // gs of the previous step no longer read
#pragma unroll
    for (int u = 0; u < MAXL; ++u) {
      const int idx = threadIdx.x + u * NT;
      if (idx < NB * ldg) gs[idx] = gpre[u];
    }
    double r = rpre;
    if (p > 0) fetch(p - 1);                                // in flight while this step is computed
    __syncthreads();
    if (ra < n && j < n) {
      double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
      const int c_lo = (p + 1) * NB, c_hi = npan * NB;      // padded columns hold zeros in gs and xs_
      for (int c = c_lo; c < c_hi; c += 4) {
        s0 = fma(gs[a * ldg + c], xs_[c * NB + jj], s0);
        s1 = fma(gs[a * ldg + c + 1], xs_[(c + 1) * NB + jj], s1);
        s2 = fma(gs[a * ldg + c + 2], xs_[(c + 2) * NB + jj], s2);
        s3 = fma(gs[a * ldg + c + 3], xs_[(c + 3) * NB + jj], s3);
      }
      r -= (s0 + s1) + (s2 + s3);
    } else {
      r = 0.0;
    }
    rblk[a * NB + jj] = r;
    __syncthreads();
    double x = 0.0;
    const double* Tp = ts + (size_t)p * NT;
    if (ra < n) {
#pragma unroll
      for (int c = 0; c < NB; ++c) x = fma(Tp[a * NB + c], rblk[c * NB + jj], x);   // T_p upper triangular (zeros below)
      if (j < n) X[(long long)ra * n + j] = x;
    }
    xs_[ra * NB + jj] = x;                                  // padded rows: zero
  }
}

// Vt[c][r] = V[r][c]  (rows x n -> n x rows), 32 x 32 tiles through shared memory
__global__ void transpose_tall_kernel(const double* __restrict__ V, long long rows, int n, double* __restrict__ Vt) {
  __shared__ double tile[32][33];
  const long long r0 = (long long)blockIdx.x * 32; const int c0 = blockIdx.y * 32;
  for (int i = threadIdx.y; i < 32; i += blockDim.y) {
    long long r = r0 + i; int c = c0 + threadIdx.x;
    tile[i][threadIdx.x] = (r < rows && c < n) ? V[r * n + c] : 0.0;
  }
  __syncthreads();
  for (int i = threadIdx.y; i < 32; i += blockDim.y) {
    int c = c0 + i; long long r = r0 + threadIdx.x;
    if (c < n && r < rows) Vt[(long long)c * rows + r] = tile[threadIdx.x][i];
  }
}

}  // namespace qk
