// K2, fast path: CholeskyQR2 of the reduced corner c~ (rows x n, n <= CHOL_MAX_N), "(unpivoted) QR".
//
//   G1 = X^T X,  R1 = chol(G1)^T,  Q1 = X R1^-1;   G2 = Q1^T Q1,  R2 = chol(G2)^T,  Q = Q1 R2^-1,  R = R2 R1.
//
// Reading A7: with full column rank the QR factorisation with diag(R) > 0 is unique, so any algorithm
// that reproduces it to rounding x cond(c~) is "the" unpivoted QR; Cholesky factors have a positive diagonal by
// construction, so no sign fix is needed.  The second pass makes Q orthonormal to O(eps) whenever
// ||Q1^T Q1 - I|| is small (cond(c~)^2 eps << 1); this kernel measures that deviation and reports it, and the host
// side falls back to the Householder path (qr_f64.cuh) when it is not small or a pivot breaks down (rank-deficient
// c~, hazard H1).  All the O(rows n^2) work runs on the DMMA GEMM; what is left here is the n x n factorisation:
//
// chol_inv_kernel: ONE CTA factors G = L L^T (n <= 208) and inverts L, entirely in shared memory.
//   * storage: the lower block triangle in 16-row block rows, block row I dense 16 x 16(I+1) with row stride
//     S_I = 16(I+1) + 4 doubles -- S_I = 4 (mod 16) makes the m8n8k4 fragment loads (8 rows x 4 columns of 8-byte
//     elements) bank-conflict free; 193 KB at n = 208.  Rows / columns beyond n are padded with the identity.
//   * blocked right-looking Cholesky, block 16: the diagonal block by ONE warp with the rows in registers (lane =
//     row, column broadcast by shuffles, rsqrt instead of sqrt + divide: ~1 us per block), the panel below it by one
//     thread per row (substitution against the 16 x 16 factor, broadcast reads), the trailing update
//     C -= L_panel L_panel^T as FP64 tensor-core tiles (mma.sync m8n8k4, SASS DMMA) straight from shared memory,
//     one 16 x 16 output block per warp.
//   * inverse M = L^-1 in place, block row by block row: M_II by one warp (lane = column), then
//     M_IJ = -sum_K (M_II L_IK) M_KJ as DMMA tiles.
//   * outputs: Rup = L^T (upper, zeros below), Llow = L, Rinv = M^T = R^-1 (upper), status / deviation.
// Deterministic: fixed summation orders, no atomics.
#pragma once
#include <cooperative_groups.h>

#include "gemm_f64.cuh"
#include "kernels_misc.cuh"

namespace qk {

constexpr int CHOL_MAX_N = 208;
constexpr int CHOL_NT = 512;

__host__ __device__ inline int chol_base(int I) { return 128 * I * (I + 1) + 64 * I; }     // doubles before block row I
__host__ __device__ inline int chol_stride(int I) { return 16 * (I + 1) + 4; }
__host__ __device__ inline size_t chol_smem_bytes(int n) {
  const int nb = (n + 15) / 16;
  return sizeof(double) * ((size_t)chol_base(nb) + 16 * nb + 64);
}

// status[0]: 0 ok, 1 = a pivot was not positive / not finite (breakdown).  dev[0] = ||G - I||_F (pass 2: the loss
// of orthogonality of Q1).  prev_status (may be null): status word of the first pass; verdict (may be null):
// verdict[0] = 1 when the CholeskyQR2 result must be discarded (either pass broke down or dev > dev_max).
// (body: CHOL_NT threads of one CTA; sm = chol_smem_bytes(n) of shared memory; every pointer may be global or shared)
constexpr double kCholFastDsum = 1e-18;   // ||Q1^T Q1 - I||_F^2 below which pass 2 takes the first-order factor

__device__ __forceinline__ void
chol_inv_body(double* sm, const double* G, int n, double* Rup, double* Llow, double* Rinv, int* status, double* dev,
              const int* prev_status, int* verdict, double dev_max,
              long long* prof /* null, or 8 cycle counters of the phases (thread 0) */,
              double fast_dsum = 0.0 /* > 0: first-order factor when ||G - I||_F^2 <= fast_dsum (see below) */) {
  const int nb = (n + 15) / 16, np = nb * 16;
  double* rd = sm + chol_base(nb);             // reciprocal diagonal of L
  double* red = rd + 16 * nb;                  // 33 doubles for the block reduction + flags
  __shared__ int bad;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int lr = lane >> 2, lc = lane & 3;
  constexpr int NW = CHOL_NT / 32;
  if (tid == 0) bad = 0;
  __syncthreads();
  long long tp[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tc = 0;
#define CHOL_TICK(i) do { if (prof && tid == 0) { const long long t_ = clock64(); tp[i] += t_ - tc; tc = t_; } } while (0)
  if (prof && tid == 0) tc = clock64();

  // ---- load the lower block triangle (identity padding), accumulate ||G - I||_F^2 over the full matrix
  double dsum = 0.0;
  for (int i = warp; i < np; i += NW) {                 // one warp per row, lanes along the row; the row's (up to 7)
    const int I = i >> 4, w = 16 * (I + 1);             // loads per lane are issued together
    double* rowp = sm + chol_base(I) + (i & 15) * chol_stride(I);
    double v[(CHOL_MAX_N + 31) / 32];
#pragma unroll
    for (int t = 0; t < (CHOL_MAX_N + 31) / 32; ++t) {
      const int j = lane + 32 * t;
      v[t] = (i == j) ? 1.0 : 0.0;
      if (j < w && i < n && j < n) v[t] = G[(long long)i * n + j];
    }
#pragma unroll
    for (int t = 0; t < (CHOL_MAX_N + 31) / 32; ++t) {
      const int j = lane + 32 * t;
      if (j < w) {
        if (i < n && j <= i) { const double d = v[t] - (i == j ? 1.0 : 0.0); dsum += (i == j ? 1.0 : 2.0) * d * d; }
        rowp[j] = v[t];
      }
    }
  }
  dsum = block_sum(dsum, red);
  CHOL_TICK(0);

  // ---- second pass of CholeskyQR2: G = Q1^T Q1 = I + E with ||E||_F ~ cond(X)^2 eps (1e-15 ... 1e-11 on the step's c~).
  // For ||E||_F <= 1e-9 the first-order factor R = I + U, R^-1 = I - U, U = striu(E) + diag(E) / 2 (U + U^T = E) is the
  // Cholesky factor to rounding -- the neglected terms are O(||E||^2) <= 1e-18 -- so the serial factorisation and
  // inversion below (most of this kernel's time) are skipped.  The branch is uniform (dsum is a block-wide sum).
  if (fast_dsum > 0.0 && dsum <= fast_dsum) {
    for (int i = warp; i < n; i += NW)
      for (int j = lane; j < n; j += 32) {
        const int hi = i > j ? i : j, lo = i > j ? j : i;        // the stored lower triangle holds G[hi][lo]
        const double g = sm[chol_base(hi >> 4) + (hi & 15) * chol_stride(hi >> 4) + lo];
        const double u = i == j ? 0.5 * (g - 1.0) : g;
        if (Llow) Llow[i * n + j] = j < i ? u : (j == i ? 1.0 + u : 0.0);
        if (Rup) Rup[i * n + j] = j > i ? u : (j == i ? 1.0 + u : 0.0);
        Rinv[i * n + j] = j > i ? -u : (j == i ? 1.0 - u : 0.0);
      }
    if (tid == 0) {
      status[0] = 0;
      dev[0] = sqrt(dsum);
      if (verdict) verdict[0] = (prev_status && prev_status[0]) ? 1 : 0;
      if (prof) for (int i = 0; i < 8; ++i) prof[i] = tp[i];
    }
    return;
  }

  // ---- blocked right-looking Cholesky with a one-block look-ahead: after the panel of block column J, warp 0 updates
  // only the next diagonal block and factors it at once (a chain of 16 dependent rsqrt, ~2 us) while the other warps do
  // the rest of the trailing update, so the diagonal-block chain is off the critical path
  auto factor_diag = [&](int J) {                       // warp 0
    const int SJ = chol_stride(J);
    double* dblk = sm + chol_base(J) + 16 * J;          // diagonal block (row stride SJ)
    const int r = lane & 15;                            // lanes 16..31 mirror lanes 0..15 (keeps the shuffles full-warp)
    double a[16];
#pragma unroll
    for (int c = 0; c < 16; ++c) a[c] = dblk[r * SJ + c];
    int brk = 0;
#pragma unroll
    for (int c = 0; c < 16; ++c) {
      double dcc = __shfl_sync(0xffffffffu, a[c], c);
      if (!(dcc > 0.0) || !(dcc < INFINITY)) { brk = 1; dcc = 1.0; }
      // the trailing columns take the UNSCALED column c times 1 / d_cc, so that their shuffles and products do not
      // wait for the reciprocal square root: the dependent chain per column is shuffle -> rsqrt -> square -> one FMA
      double t[16];
#pragma unroll
      for (int c2 = c + 1; c2 < 16; ++c2) t[c2] = a[c] * __shfl_sync(0xffffffffu, a[c], c2);   // a[r][c] a[c2][c]
      const double rs = rsqrt(dcc);
      const double rs2 = rs * rs;
#pragma unroll
      for (int c2 = c + 1; c2 < 16; ++c2) a[c2] = fma(-t[c2], rs2, a[c2]);   // a[r][c2] -= l[r][c] l[c2][c]   (used for r >= c2)
      a[c] = (r == c) ? dcc * rs : a[c] * rs;            // l[r][c] for r >= c (rows above: unused)
      if (lane == c) rd[16 * J + c] = rs;
    }
    if (lane < 16) {
#pragma unroll
      for (int c = 0; c < 16; ++c) dblk[r * SJ + c] = (c <= r) ? a[c] : 0.0;
    }
    if (brk && lane == 0) bad = 1;
  };
  // C[I2][J2] -= L[I2][J] L[J2][J]^T, block number q of the trailing triangle (row by row), one warp
  auto update_block = [&](int J, int q) {
    int ri = (int)((sqrtf(8.0f * q + 1.0f) - 1.0f) * 0.5f);
    while ((ri + 1) * (ri + 2) / 2 <= q) ++ri;
    while (ri * (ri + 1) / 2 > q) --ri;
    const int cj = q - ri * (ri + 1) / 2;
    const int I2 = J + 1 + ri, J2 = J + 1 + cj;
    const int SI = chol_stride(I2), S2 = chol_stride(J2);
    const double* ap = sm + chol_base(I2) + lr * SI + 16 * J + lc;
    const double* bp = sm + chol_base(J2) + lr * S2 + 16 * J + lc;
    double* cp = sm + chol_base(I2) + lr * SI + 16 * J2 + 2 * lc;
    double acc[2][2][2];
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
      for (int ni = 0; ni < 2; ++ni) {
        const double2 t = *reinterpret_cast<const double2*>(cp + mi * 8 * SI + ni * 8);
        acc[mi][ni][0] = t.x; acc[mi][ni][1] = t.y;
      }
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      const double a0 = -ap[ks * 4], a1 = -ap[8 * SI + ks * 4];
      const double b0 = bp[ks * 4], b1 = bp[8 * S2 + ks * 4];
      dmma884(acc[0][0][0], acc[0][0][1], a0, b0);
      dmma884(acc[0][1][0], acc[0][1][1], a0, b1);
      dmma884(acc[1][0][0], acc[1][0][1], a1, b0);
      dmma884(acc[1][1][0], acc[1][1][1], a1, b1);
    }
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
      for (int ni = 0; ni < 2; ++ni)
        *reinterpret_cast<double2*>(cp + mi * 8 * SI + ni * 8) = make_double2(acc[mi][ni][0], acc[mi][ni][1]);
  };
  for (int J = -1; J < nb; ++J) {                       // J = -1: only the first diagonal block
    if (J >= 0) {
      const int SJ = chol_stride(J);
      const double* dblk = sm + chol_base(J) + 16 * J;
      // panel below the diagonal block: row i solves x L_JJ^T = a  (one thread per row)
      const int nrow = np - 16 * (J + 1);
      if (tid < nrow) {
        const int i = 16 * (J + 1) + tid, I = i >> 4;
        double* row = sm + chol_base(I) + (i & 15) * chol_stride(I) + 16 * J;
        double x[16];
#pragma unroll
        for (int c = 0; c < 16; c += 2) { const double2 t = *reinterpret_cast<const double2*>(row + c); x[c] = t.x; x[c + 1] = t.y; }
#pragma unroll
        for (int c = 0; c < 16; ++c) {
          x[c] *= rd[16 * J + c];
#pragma unroll
          for (int c2 = c + 1; c2 < 16; ++c2) x[c2] = fma(-x[c], dblk[c2 * SJ + c], x[c2]);
        }
#pragma unroll
        for (int c = 0; c < 16; c += 2) *reinterpret_cast<double2*>(row + c) = make_double2(x[c], x[c + 1]);
      }
      __syncthreads();
      CHOL_TICK(2);
    }
    const int nr = nb - J - 1, nt = J >= 0 ? nr * (nr + 1) / 2 : 0;
    if (warp == 0) {
      if (J < 0 || nt > 0) {
        if (J >= 0) update_block(J, 0);
        __syncwarp();
        factor_diag(J + 1);
      }
    } else {
      for (int q = warp; q < nt; q += NW - 1) update_block(J, q);
    }
    __syncthreads();
    CHOL_TICK(3);
  }

  // ---- write L (lower) and R = L^T (upper)
  for (int i = warp; i < n; i += NW) {                  // one warp per row, coalesced stores; R[i][j] = L[j][i]
    const double* Li = sm + chol_base(i >> 4) + (i & 15) * chol_stride(i >> 4);
    for (int j = lane; j < n; j += 32) {
      if (Llow) Llow[i * n + j] = j <= i ? Li[j] : 0.0;
      if (Rup) Rup[i * n + j] = j >= i ? sm[chol_base(j >> 4) + (j & 15) * chol_stride(j >> 4) + i] : 0.0;
    }
  }
  if (tid == 0) {
    status[0] = bad;
    dev[0] = sqrt(dsum);
    if (verdict) verdict[0] = (bad || (prev_status && prev_status[0]) || !(sqrt(dsum) <= dev_max)) ? 1 : 0;
  }
  __syncthreads();
  CHOL_TICK(4);

  // ---- M = L^-1 in place.  Diagonal blocks first: warp I, lane = column c of inv(L_II).
  for (int I = warp; I < nb; I += NW) {
    const int S = chol_stride(I);
    double* dblk = sm + chol_base(I) + 16 * I;
    const int c = lane & 15;
    double x[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) x[r] = 0.0;              // x[r] accumulates -sum_k L[r][k] x[k] until row r is finalised
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      const double xr = (r == c ? 1.0 : x[r]) * rd[16 * I + r];      // rows above c stay 0
      x[r] = r >= c ? xr : 0.0;
#pragma unroll
      for (int r2 = r + 1; r2 < 16; ++r2) x[r2] = fma(-dblk[r2 * S + r], x[r], x[r2]);
    }
    __syncwarp();
    if (lane < 16) {
#pragma unroll
      for (int r = 0; r < 16; ++r) dblk[r * S + c] = x[r];
    }
  }
  __syncthreads();
  CHOL_TICK(5);
  for (int I = 1; I < nb; ++I) {
    const int SI = chol_stride(I);
    double* rowI = sm + chol_base(I);
    // P0: L'_IK = M_II L_IK for K < I (in place; a warp touches only its own block and reads the diagonal block)
    for (int K = warp; K < I; K += NW) {
      const double* ap = rowI + lr * SI + 16 * I + lc;               // A = M_II
      const double* bp = rowI + lc * SI + 16 * K + lr;               // B[k][n] = L_IK[k][n]
      double acc[2][2][2];
#pragma unroll
      for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 2; ++ni) acc[mi][ni][0] = acc[mi][ni][1] = 0.0;
#pragma unroll
      for (int ks = 0; ks < 4; ++ks) {
        const double a0 = ap[ks * 4], a1 = ap[8 * SI + ks * 4];
        const double b0 = bp[ks * 4 * SI], b1 = bp[ks * 4 * SI + 8];
        dmma884(acc[0][0][0], acc[0][0][1], a0, b0);
        dmma884(acc[0][1][0], acc[0][1][1], a0, b1);
        dmma884(acc[1][0][0], acc[1][0][1], a1, b0);
        dmma884(acc[1][1][0], acc[1][1][1], a1, b1);
      }
      __syncwarp();
      double* cp = rowI + lr * SI + 16 * K + 2 * lc;
#pragma unroll
      for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 2; ++ni)
          *reinterpret_cast<double2*>(cp + mi * 8 * SI + ni * 8) = make_double2(acc[mi][ni][0], acc[mi][ni][1]);
    }
    __syncthreads();
    // P1: acc_J = sum_{K=J}^{I-1} L'_IK M_KJ   (rows K < I already hold M); P2: M_IJ = -acc_J
    double acc[2][2][2];
    const int Jw = warp;                                             // nb <= 13 <= NW: one block column per warp
    if (Jw < I) {
#pragma unroll
      for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 2; ++ni) acc[mi][ni][0] = acc[mi][ni][1] = 0.0;
      for (int K = Jw; K < I; ++K) {
        const int SK = chol_stride(K);
        const double* ap = rowI + lr * SI + 16 * K + lc;
        const double* bp = sm + chol_base(K) + lc * SK + 16 * Jw + lr;
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
          const double a0 = ap[ks * 4], a1 = ap[8 * SI + ks * 4];
          const double b0 = bp[ks * 4 * SK], b1 = bp[ks * 4 * SK + 8];
          dmma884(acc[0][0][0], acc[0][0][1], a0, b0);
          dmma884(acc[0][1][0], acc[0][1][1], a0, b1);
          dmma884(acc[1][0][0], acc[1][0][1], a1, b0);
          dmma884(acc[1][1][0], acc[1][1][1], a1, b1);
        }
      }
    }
    __syncthreads();
    if (Jw < I) {
      double* cp = rowI + lr * SI + 16 * Jw + 2 * lc;
#pragma unroll
      for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 2; ++ni)
          *reinterpret_cast<double2*>(cp + mi * 8 * SI + ni * 8) = make_double2(-acc[mi][ni][0], -acc[mi][ni][1]);
    }
    // (the next P0 touches block row I+1 only; its closing barrier orders these stores before the next P1)
  }
  __syncthreads();
  CHOL_TICK(6);
  // ---- R^-1 = M^T (upper)
  for (int r = warp; r < n; r += NW)                    // R^-1[r][c] = M[c][r], M = L^-1
    for (int c = lane; c < n; c += 32)
      Rinv[r * n + c] = c >= r ? sm[chol_base(c >> 4) + (c & 15) * chol_stride(c >> 4) + r] : 0.0;
  if (prof) {
    __syncthreads();
    CHOL_TICK(7);
    if (tid == 0) for (int i = 0; i < 8; ++i) prof[i] = tp[i];
  }
#undef CHOL_TICK
}

__global__ void __launch_bounds__(CHOL_NT, 1)
chol_inv_kernel(const double* __restrict__ G, int n, double* __restrict__ Rup, double* __restrict__ Llow,
                double* __restrict__ Rinv, int* __restrict__ status, double* __restrict__ dev,
                const int* __restrict__ prev_status, int* __restrict__ verdict, double dev_max,
                long long* __restrict__ prof, double fast_dsum = 0.0) {
  extern __shared__ __align__(16) double sm[];
  chol_inv_body(sm, G, n, Rup, Llow, Rinv, status, dev, prev_status, verdict, dev_max, prof, fast_dsum);
}

// ------------------------------------------------------------------------------------------------------------------
// CholeskyQR2 of a small c~ (n <= CHOLC_MAX_N columns, rows <= 16 slabs that fit shared memory: cfg1, cfg2) as ONE
// launch of one thread-block cluster instead of eleven dependent launches (which cost 10-20 us each at these sizes:
// K2 was 55 % of the cfg1 / cfg2 step).  The rows of X are dealt out to the CTAs in contiguous slabs that stay in
// shared memory through both passes; per pass: local Gram matrix of the slab -> fixed-order sum over the cluster
// through distributed shared memory (every CTA ends with the full G) -> every CTA factors and inverts G redundantly
// (chol_inv_body) -> slab <- slab R^-1.  Rank 0 writes R = L2^T R1 and the status / verdict words.  Deterministic.
constexpr int CHOLC_MAX_N = 64;
// slab pitch: >= n, = 4 (mod 16) doubles, so that the m8n8k4 fragment loads of both products are conflict-free (as in the
// Cholesky kernel's block rows); slab rows padded to a multiple of 8 (zero rows: they complete the last fragments)
__host__ __device__ inline int cholqr2_slab_pitch(int n) { return ((n + 11) / 16) * 16 + 4; }
__host__ __device__ inline size_t cholqr2_cluster_smem_bytes(int n, int rpc) {
  const size_t rp = (size_t)((rpc + 7) & ~7);
  return sizeof(double) * ((size_t)4 * n * n + 2 * rp * cholqr2_slab_pitch(n) + 8) + chol_smem_bytes(n);
}

__global__ void __launch_bounds__(CHOL_NT, 1)
cholqr2_cluster_kernel(const double* __restrict__ X, long long rows, int n, double* __restrict__ Q, double* __restrict__ R,
                       int* __restrict__ cstat /* [3] */, double* __restrict__ cdev /* [2] */, double dev_max, int rpc,
                       long long* __restrict__ prof /* null, or 8 cycle counters of rank 0's phases */) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  extern __shared__ __align__(16) double csm[];
  const int nn = n * n;
  double* Gp = csm;                      // my slab's partial Gram matrix (pass 2: reused for L2 after the sum)
  double* Gf = Gp + nn;                  // the full Gram matrix (written by all ranks)
  double* R1 = Gf + nn;                  // R of pass 1
  double* Ri = R1 + nn;                  // R^-1 of the current pass
  const int P = cholqr2_slab_pitch(n), rp = (rpc + 7) & ~7;
  double* Xs = Ri + nn;                  // rp x P: my rows of X, then of Q1 after the swap (pad rows / columns zero)
  double* Ys = Xs + (size_t)rp * P;
  double* sc = Ys + (size_t)rp * P;      // [0..1] deviations, ints behind
  int* st = reinterpret_cast<int*>(sc + 4);
  double* ws = sc + 8;                   // chol_inv_body's workspace
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int lr = lane >> 2, lc = lane & 3;
  constexpr int NW = CHOL_NT / 32;
  long long tp[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tc = 0;
#define CQ_TICK(i) do { if (prof && tid == 0 && rank == 0) { const long long t_ = clock64(); tp[i] += t_ - tc; tc = t_; } } while (0)
  if (prof && tid == 0 && rank == 0) tc = clock64();
  const long long r0 = (long long)rank * rpc;
  const int rl = (int)(rows - r0 < 0 ? 0 : (rows - r0 < rpc ? rows - r0 : rpc));      // my rows
  for (int i = tid; i < rp * P; i += CHOL_NT) {
    const int r = i / P, c = i - r * P;
    Xs[i] = (r < rl && c < n) ? X[(r0 + r) * n + c] : 0.0;
    Ys[i] = 0.0;
  }
  __syncthreads();
  CQ_TICK(0);
  double* src = Xs;
  double* dst = Ys;
  const int nf = (n + 7) >> 3;             // 8-wide fragment columns
  const int nrf = (rl + 7) >> 3;           // 8-row fragments of my slab
  for (int pass = 0; pass < 2; ++pass) {
    // local Gram matrix of the slab as DMMA tiles straight from shared memory: 8 x 8 output fragments of the lower
    // fragment triangle, up to three per warp in flight; G[i][j] = sum_r X[r][i] X[r][j]: both operands are read as
    // src[(r + lc) * P + col + lr] (conflict-free for P = 4 mod 16); the pad rows are zero
    {
      const int nfr = nf * (nf + 1) / 2;
      for (int q0 = warp; q0 < nfr; q0 += 3 * NW) {
        int i0[3], j0[3];
        double acc[3][2];
#pragma unroll
        for (int t = 0; t < 3; ++t) {
          int q = q0 + t * NW; if (q >= nfr) q = q0;           // a duplicate of the first fragment (not stored)
          int fi = (int)((sqrtf(8.0f * q + 1.0f) - 1.0f) * 0.5f);
          while ((fi + 1) * (fi + 2) / 2 <= q) ++fi;
          while (fi * (fi + 1) / 2 > q) --fi;
          i0[t] = fi << 3; j0[t] = (q - fi * (fi + 1) / 2) << 3;
          acc[t][0] = acc[t][1] = 0.0;
        }
        const double* sp = src + lc * P + lr;
        for (int r = 0; r < 8 * nrf; r += 4) {
#pragma unroll
          for (int t = 0; t < 3; ++t) dmma884(acc[t][0], acc[t][1], sp[r * P + i0[t]], sp[r * P + j0[t]]);
        }
#pragma unroll
        for (int t = 0; t < 3; ++t) {
          if (q0 + t * NW < nfr) {
            const int i = i0[t] + lr, j = j0[t] + 2 * lc;
            if (i < n && j < n) Gp[i * n + j] = acc[t][0];
            if (i < n && j + 1 < n) Gp[i * n + j + 1] = acc[t][1];
          }
        }
      }
    }
    const int nq = (n + 3) >> 2, nblk = nq * (nq + 1) / 2;
    CQ_TICK(1);
    cluster.sync();
    CQ_TICK(2);
    // fixed-order sum over the ranks of the lower block triangle; rank r owns the blocks q = r (mod C) and hands the
    // sums to everybody; the upper triangle is mirrored locally afterwards
    for (int w = rank * 16 + C * 16 * (tid >> 4) + (tid & 15); (w >> 4) < nblk; w += C * 16 * (CHOL_NT >> 4)) {
      const int q = w >> 4, el = w & 15;
      int bi = (int)((sqrtf(8.0f * q + 1.0f) - 1.0f) * 0.5f);
      while ((bi + 1) * (bi + 2) / 2 <= q) ++bi;
      while (bi * (bi + 1) / 2 > q) --bi;
      const int bj = q - bi * (bi + 1) / 2, i = (bi << 2) + (el >> 2), j = (bj << 2) + (el & 3);
      if (i < n && j < n) {
        const int e = i * n + j;
        double s = 0.0;
        for (int qq = 0; qq < C; ++qq) s += cluster.map_shared_rank(Gp, qq)[e];
        for (int qq = 0; qq < C; ++qq) cluster.map_shared_rank(Gf, qq)[e] = s;
      }
    }
    CQ_TICK(3);
    cluster.sync();
    CQ_TICK(2);
    for (int e = tid; e < nn; e += CHOL_NT) {               // mirror: blocks above the block diagonal
      const int i = e / n, j = e % n;
      if ((j >> 2) > (i >> 2)) Gf[e] = Gf[j * n + i];
    }
    __syncthreads();
    if (pass == 0) chol_inv_body(ws, Gf, n, R1, nullptr, Ri, st, sc, nullptr, nullptr, 0.0, nullptr);
    else           chol_inv_body(ws, Gf, n, nullptr, Gp, Ri, st + 1, sc + 1, st, st + 2, dev_max, nullptr, kCholFastDsum);
    __syncthreads();
    CQ_TICK(4);
    // slab <- slab R^-1 (R^-1 upper triangular: k <= c) as DMMA tiles: a work item is one fragment column and up to four
    // row fragments, the B fragment of a k-step is loaded once for the four; pass 1 into the other buffer, pass 2 to Q
    {
      const int nrg = (nrf + 3) >> 2;
      for (int it = warp; it < nf * nrg; it += NW) {
        const int cf = it / nrg, rg = it - cf * nrg, c0 = cf << 3, rf0 = rg << 2;
        double acc[4][2];
#pragma unroll
        for (int t = 0; t < 4; ++t) acc[t][0] = acc[t][1] = 0.0;
        const int kend = c0 + 8 < n ? c0 + 8 : n;           // R^-1[k][c] = 0 for k > c
        const double* ap = src + (size_t)(rf0 * 8 + lr) * P + lc;
        for (int k = 0; k < kend; k += 4) {
          const int kk = k + lc, cc = c0 + lr;
          const double bv = (kk < n && cc < n) ? Ri[kk * n + cc] : 0.0;
#pragma unroll
          for (int t = 0; t < 4; ++t)
            if (rf0 + t < nrf) dmma884(acc[t][0], acc[t][1], ap[(size_t)t * 8 * P + k], bv);
        }
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          const int r = (rf0 + t) * 8 + lr, c = c0 + 2 * lc;
          if (rf0 + t < nrf && r < rl) {
            if (pass == 0) { if (c < n) dst[r * P + c] = acc[t][0]; if (c + 1 < n) dst[r * P + c + 1] = acc[t][1]; }
            else { if (c < n) Q[(r0 + r) * n + c] = acc[t][0]; if (c + 1 < n) Q[(r0 + r) * n + c + 1] = acc[t][1]; }
          }
        }
      }
    }
    __syncthreads();
    CQ_TICK(5);
    double* t = src; src = dst; dst = t;
  }
  // R = R2 R1 = L2^T R1 (both triangular: j runs over i..k): every rank holds L2 and R1, rank r writes the rows i = r (mod C)
  for (int e = tid; e < ((n - rank + C - 1) / C) * n; e += CHOL_NT) {
    const int i = rank + C * (e / n), k = e % n;
    double s = 0.0;
    for (int j = i; j <= k; ++j) s = fma(Gp[j * n + i], R1[j * n + k], s);
    R[i * n + k] = s;
  }
  if (rank == 0) {
    if (tid == 0) { cstat[0] = st[0]; cstat[1] = st[1]; cstat[2] = st[2]; cdev[0] = sc[0]; cdev[1] = sc[1]; }
    if (prof) {
      __syncthreads();
      CQ_TICK(6);
      if (tid == 0) for (int i = 0; i < 8; ++i) prof[i] = tp[i];
    }
  }
#undef CQ_TICK
}

// The conditional-graph hook of the fallback: 1 = run the body (the Householder path).
__global__ void cholqr_set_cond_kernel(cudaGraphConditionalHandle hnd, const int* __restrict__ verdict) {
  if (threadIdx.x == 0) cudaGraphSetConditional(hnd, verdict[0] ? 1u : 0u);
}

}  // namespace qk
