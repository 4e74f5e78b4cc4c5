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
__global__ void __launch_bounds__(CHOL_NT, 1)
chol_inv_kernel(const double* __restrict__ G, int n, double* __restrict__ Rup, double* __restrict__ Llow,
                double* __restrict__ Rinv, int* __restrict__ status, double* __restrict__ dev,
                const int* __restrict__ prev_status, int* __restrict__ verdict, double dev_max,
                long long* __restrict__ prof /* null, or 8 cycle counters of the phases (thread 0) */) {
  extern __shared__ __align__(16) double sm[];
  const int nb = (n + 15) / 16, np = nb * 16;
  double* rd = sm + chol_base(nb);             // reciprocal diagonal of L
  double* red = rd + 16 * nb;                  // 33 doubles for the block reduction + flags
  __shared__ int bad;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int lr = lane >> 2, lc = lane & 3;
  constexpr int NW = CHOL_NT / 32;
  if (tid == 0) bad = 0;
  long long tp[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tc = 0;
#define CHOL_TICK(i) do { if (prof && tid == 0) { const long long t_ = clock64(); tp[i] += t_ - tc; tc = t_; } } while (0)
  if (prof && tid == 0) tc = clock64();

  // ---- load the lower block triangle (identity padding), accumulate ||G - I||_F^2 over the full matrix
  double dsum = 0.0;
  for (int I = 0; I < nb; ++I) {
    const int w = 16 * (I + 1), S = chol_stride(I);
    double* blk = sm + chol_base(I);
    for (int e = tid; e < 16 * w; e += CHOL_NT) {
      const int r = e / w, j = e % w, i = 16 * I + r;
      double v = (i == j) ? 1.0 : 0.0;
      if (i < n && j < n) {
        v = G[(long long)i * n + j];
        if (j <= i) { const double t = v - (i == j ? 1.0 : 0.0); dsum += (i == j ? 1.0 : 2.0) * t * t; }
      }
      blk[r * S + j] = v;
    }
  }
  dsum = block_sum(dsum, red);
  CHOL_TICK(0);

  // ---- blocked right-looking Cholesky
  for (int J = 0; J < nb; ++J) {
    const int SJ = chol_stride(J);
    double* dblk = sm + chol_base(J) + 16 * J;          // diagonal block (row stride SJ)
    if (warp == 0) {
      const int r = lane & 15;                          // lanes 16..31 mirror lanes 0..15 (keeps the shuffles full-warp)
      double a[16];
#pragma unroll
      for (int c = 0; c < 16; ++c) a[c] = dblk[r * SJ + c];
      int brk = 0;
#pragma unroll
      for (int c = 0; c < 16; ++c) {
        double dcc = __shfl_sync(0xffffffffu, a[c], c);
        if (!(dcc > 0.0) || !(dcc < INFINITY)) { brk = 1; dcc = 1.0; }
        const double rs = rsqrt(dcc);
        a[c] = (r == c) ? dcc * rs : a[c] * rs;          // l[r][c] for r >= c (rows above: unused)
        if (lane == c) rd[16 * J + c] = rs;
#pragma unroll
        for (int c2 = c + 1; c2 < 16; ++c2) {
          const double l2 = __shfl_sync(0xffffffffu, a[c], c2);     // l[c2][c]
          a[c2] = fma(-a[c], l2, a[c2]);                             // a[r][c2] -= l[r][c] l[c2][c]   (used for r >= c2)
        }
      }
      if (lane < 16) {
#pragma unroll
        for (int c = 0; c < 16; ++c) dblk[r * SJ + c] = (c <= r) ? a[c] : 0.0;
      }
      if (brk && lane == 0) bad = 1;
    }
    __syncthreads();
    CHOL_TICK(1);
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
    // trailing update: C[I2][J2] -= L[I2][J] L[J2][J]^T for J < J2 <= I2 < nb, one 16 x 16 block per warp
    const int nr = nb - J - 1, nt = nr * (nr + 1) / 2;
    for (int q = warp; q < nt; q += NW) {
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
    }
    __syncthreads();
    CHOL_TICK(3);
  }

  // ---- write L (lower) and R = L^T (upper)
  for (int idx = tid; idx < n * n; idx += CHOL_NT) {
    const int i = idx / n, j = idx % n;
    if (Llow) Llow[idx] = j <= i ? sm[chol_base(i >> 4) + (i & 15) * chol_stride(i >> 4) + j] : 0.0;
    if (Rup) Rup[idx] = i <= j ? sm[chol_base(j >> 4) + (j & 15) * chol_stride(j >> 4) + i] : 0.0;
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
  for (int idx = tid; idx < n * n; idx += CHOL_NT) {
    const int r = idx / n, c = idx % n;
    Rinv[idx] = r <= c ? sm[chol_base(c >> 4) + (c & 15) * chol_stride(c >> 4) + r] : 0.0;
  }
  if (prof) {
    __syncthreads();
    CHOL_TICK(7);
    if (tid == 0) for (int i = 0; i < 8; ++i) prof[i] = tp[i];
  }
#undef CHOL_TICK
}

// The conditional-graph hook of the fallback: 1 = run the body (the Householder path).
__global__ void cholqr_set_cond_kernel(cudaGraphConditionalHandle hnd, const int* __restrict__ verdict) {
  if (threadIdx.x == 0) cudaGraphSetConditional(hnd, verdict[0] ? 1u : 0u);
}

}  // namespace qk
