// FP64 tensor-core GEMM for the QR-CTMRG contractions (K1, K2b, K2c, K3, K4, K5, K6).
//
//   out[ro(i) + co(j)] (op)= sum_k opA(i,k) * B[k*ldb + j]      i < M, j < N, k < K
//
// * B is always K x N row-major (N contiguous).
// * opA: transA = 1 -> A stored K x M (M contiguous), the form every large
//   contraction of the step takes once the producers write their outputs in the
//   layout the consumer wants; transA = 0 -> A stored M x K.
// * ro/co are two-level strided index maps, so the leg permutations between the
//   contractions of (E3) are fused into the epilogue of the producing GEMM:
//       ro(i) = (i / rdiv) * rs_hi + (i % rdiv) * rs_lo     (same for co)
// * math: mma.sync.aligned.m8n8k4 f64 (SASS DMMA.8x8x4), the only FP64 tensor
//   instruction sm_100a has (tcgen05 has no f64 kind).  Two kernels: gemm_f64_dmma
//   (small / unaligned cases: a 4-stage cp.async (LDGSTS) ring, zero-filled at the
//   ragged edges) and gemm_f64_dmma_ws (every large contraction: a TMA producer warp
//   feeding an mbarrier ring, see below).  Shared-memory rows are padded by 4 doubles
//   so both fragment loads are conflict free.
// * K splitting, all deterministic (fixed summation order, no atomics): split-K
//   (gridDim.z slices write plain partial outputs, reduce_splitk sums them) and, in
//   the ws kernel, stream-K / hybrid schedules with streamk_fixup.
#pragma once
#include <cuda.h>            // CUtensorMap (type only: the encoder is reached through cudaGetDriverEntryPoint)
#include <cuda_runtime.h>
#include <stdint.h>

namespace qk {

struct IndexMap {          // idx -> (idx / div) * hi + ((idx % div) / div0) * lo + (idx % div0) * lo0
  int div;
  long long hi, lo;
  int div0 = 1;            // third level (default: none)
  long long lo0 = 0;
  __host__ __device__ long long operator()(int idx) const {
    const int r = idx % div;
    return (long long)(idx / div) * hi + (long long)(r / div0) * lo + (long long)(r % div0) * lo0;
  }
};
__host__ __device__ inline IndexMap plain_map(long long ld) { return IndexMap{1, ld, 0}; }

struct GemmArgs {
  const double* A; long long lda; int transA;
  const double* B; long long ldb;
  double* out;
  IndexMap ro, co;
  int M, N, K;
  int ktiles_per_split;      // in units of BK tiles; gridDim.z splits
  long long split_stride;    // elements between partial outputs (split-K only)
  int mode;                  // 0: out = acc, 1: out = out - acc, 2: out = out + acc
  int vecA, vecB;            // 16-byte cp.async legal for A / B
  // transA = 1 only: logical k-row r of A lives at row ka(r) of the stored matrix (default identity)
  IndexMap ka = IndexMap{1, 1, 0};
  // batched launch (gridDim.z = batch, no split-K): A += za(z) elements, out += z * zo elements
  int batch = 0;
  IndexMap za = IndexMap{1, 0, 0};
  long long zo = 0;
  int nz = 1;                // number of z slices (splits or batches) -- work list of the ws kernel
  int epi = 0;               // ws kernel epilogue: 0 = fragments straight to global, 1 = staged through shared
                             // memory so that the 32 lanes of a store run along the column index j, 2 = dense
                             // blocks: the columns come in groups of dense_wc whose 8-row blocks are contiguous in
                             // the output (row stride dense_wc); each block leaves with ONE bulk store from shared
                             // memory (cp.async.bulk.global.shared::cta, SASS UBLKCP) instead of 8 * dense_wc stores
  int dense_wc = 0, dense_magic = 0;   // epi 2: group width, ceil(65536 / dense_wc) (c / wc = c * magic >> 16, c < 128)
  // stream-K (ws kernel, nz = 1, no batch): the tiles x k-tiles units are dealt out evenly and contiguously to the
  // gridDim.x CTAs; a CTA that covers only part of a tile's k range writes a plain BM x BN partial tile to slot
  // 2 * blockIdx.x (its first segment) or 2 * blockIdx.x + 1 (its last) of sk_ws, and streamk_fixup sums the
  // partial tiles of every split tile in ascending k (fixed order).
  int sk = 0;
  int sk_t1 = 0;             // whole-tile CTAs ahead of the stream-K CTAs (hybrid schedule)
  double* sk_ws = nullptr;
  // ws kernel: tma = 1 -> the operand tiles are fetched with ONE tiled bulk tensor copy each (cp.async.bulk.tensor.2d,
  // SASS UTMALDG) through these tensor maps instead of one linear bulk copy per k-row.  The box is BK rows of
  // BM + PAD (BN + PAD) columns, i.e. it is as wide as the padded shared-memory pitch, so the dense box the copy
  // engine writes IS the conflict-free padded layout (the 4 extra columns are the neighbour tile's, never read);
  // rows beyond K and columns beyond M / N are zero-filled by the copy engine.
  int tma = 0;
  alignas(64) CUtensorMap tmA, tmB;
};

// First unit of CTA c.  The first t1 CTAs take one whole tile each (nkt units, stored directly); the remaining
// ncta - t1 CTAs share the rest of the units evenly.  t1 = 0: pure stream-K.  t1 = whole waves of tiles: only the
// ragged last wave is dealt out by k-tiles ("data-parallel + stream-K" hybrid).
__host__ __device__ inline long long sk_first_unit(long long c, long long units, long long ncta, long long t1, long long nkt) {
  if (c <= t1) return c * nkt;
  return t1 * nkt + (c - t1) * (units - t1 * nkt) / (ncta - t1);
}

constexpr int BK = 16;
constexpr int PAD = 4;

// Programmatic dependent launch: the kernels of a step are short and strictly dependent, so each one lets its
// successor in the stream be set up at once (launch_dependents: the successor's CTAs become resident as SM slots free
// up and run their own prologue) and then waits until its predecessor has completed and flushed its writes (wait).  A
// no-op for kernels launched without the programmatic-serialisation attribute.
__device__ __forceinline__ void pdl_sync() {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
}

__device__ __forceinline__ void cp_async16(void* smem, const void* g, int src_bytes) {
  uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(g), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* g, int src_bytes) {
  uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(g), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// Load a [BK][W] tile (row kk, W contiguous elements starting at column c0 of a
// row-major matrix with leading dimension ld, logical width `width`) into smem
// rows of W + PAD doubles.  Rows kk >= krows and columns >= width are zero filled.
template <int W, int NT>
__device__ __forceinline__ void load_tile_rows(double* s, const double* g, long long ld, int k0,
                                               int krows, int c0, int width, bool vec, int tid) {
  constexpr int LDS = W + PAD;
  if (vec) {
    constexpr int CH = W / 2;                       // 16-byte chunks per row
    for (int c = tid; c < BK * CH; c += NT) {
      int kk = c / CH, cc = (c % CH) * 2;
      int rem = width - (c0 + cc);
      int bytes = (kk < krows && rem > 0) ? (rem >= 2 ? 16 : 8) : 0;
      const double* src = bytes ? g + (long long)(k0 + kk) * ld + c0 + cc : g;
      cp_async16(s + kk * LDS + cc, src, bytes);
    }
  } else {
    for (int c = tid; c < BK * W; c += NT) {
      int kk = c / W, cc = c % W;
      int bytes = (kk < krows && c0 + cc < width) ? 8 : 0;
      const double* src = bytes ? g + (long long)(k0 + kk) * ld + c0 + cc : g;
      cp_async8(s + kk * LDS + cc, src, bytes);
    }
  }
}

// transA = 0: A stored [M][K]; gather a [BK][W] tile transposed (8-byte copies).
template <int W, int NT>
__device__ __forceinline__ void load_tile_cols(double* s, const double* g, long long ld, int k0,
                                               int krows, int r0, int height, int tid) {
  constexpr int LDS = W + PAD;
  for (int c = tid; c < BK * W; c += NT) {
    int mm = c / BK, kk = c % BK;                    // kk fastest -> contiguous global reads
    int bytes = (kk < krows && r0 + mm < height) ? 8 : 0;
    const double* src = bytes ? g + (long long)(r0 + mm) * ld + k0 + kk : g;
    cp_async8(s + kk * LDS + mm, src, bytes);
  }
}

template <int BM, int BN, int WM, int WN, int STAGES>
__global__ void __launch_bounds__((BM / WM) * (BN / WN) * 32, (BM >= 128 ? 1 : 2))
gemm_f64_dmma(GemmArgs p) {
  constexpr int NW_M = BM / WM, NW_N = BN / WN;
  constexpr int NT = NW_M * NW_N * 32;
  constexpr int LDA_S = BM + PAD, LDB_S = BN + PAD;
  constexpr int A_STAGE = BK * LDA_S, B_STAGE = BK * LDB_S;
  constexpr int FM = WM / 8, FN = WN / 8;
  extern __shared__ __align__(128) double smem[];
  double* As = smem;
  double* Bs = smem + STAGES * A_STAGE;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / NW_N) * WM, wn0 = (warp % NW_N) * WN;
  const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
  const int lr = lane >> 2, lc = lane & 3;

  const int nkt_total = (p.K + BK - 1) / BK;
  const int kt_begin = blockIdx.z * p.ktiles_per_split;
  int kt_end = kt_begin + p.ktiles_per_split;
  if (kt_end > nkt_total) kt_end = nkt_total;
  const int nkt = kt_end > kt_begin ? kt_end - kt_begin : 0;

  double acc[FM][FN][2];
#pragma unroll
  for (int i = 0; i < FM; ++i)
#pragma unroll
    for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
  pdl_sync();

  auto load_stage = [&](int kt, int stage) {
    int k0 = (kt_begin + kt) * BK;
    int krows = p.K - k0; if (krows > BK) krows = BK;
    if (p.transA) load_tile_rows<BM, NT>(As + stage * A_STAGE, p.A, p.lda, k0, krows, m0, p.M, p.vecA, tid);
    else          load_tile_cols<BM, NT>(As + stage * A_STAGE, p.A, p.lda, k0, krows, m0, p.M, tid);
    load_tile_rows<BN, NT>(Bs + stage * B_STAGE, p.B, p.ldb, k0, krows, n0, p.N, p.vecB, tid);
  };

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < nkt) load_stage(s, s);
    cp_async_commit();
  }
  // output offsets of the tile's rows and columns, one map evaluation per thread while the first copies are in flight
  // (a map costs two integer divisions; per fragment element they made the epilogue of a three-k-tile GEMM several
  // microseconds long)
  __shared__ long long row_off[BM], col_off[BN];
  for (int t = tid; t < BM + BN; t += NT) {
    if (t < BM) row_off[t] = (m0 + t < p.M) ? p.ro(m0 + t) : 0;
    else col_off[t - BM] = (n0 + t - BM < p.N) ? p.co(n0 + t - BM) : 0;
  }
  __syncthreads();

  for (int kt = 0; kt < nkt; ++kt) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    {
      int nxt = kt + STAGES - 1;
      if (nxt < nkt) load_stage(nxt, nxt % STAGES);
      cp_async_commit();
    }
    const double* as = As + (kt % STAGES) * A_STAGE + wm0 + lr;
    const double* bs = Bs + (kt % STAGES) * B_STAGE + wn0 + lr;
    int k0 = (kt_begin + kt) * BK;
    int ksteps = (p.K - k0 + 3) >> 2; if (ksteps > BK / 4) ksteps = BK / 4;
#pragma unroll
    for (int ks = 0; ks < BK / 4; ++ks) {
      if (ks < ksteps) {
        double af[FM], bf[FN];
#pragma unroll
        for (int i = 0; i < FM; ++i) af[i] = as[(ks * 4 + lc) * LDA_S + i * 8];
#pragma unroll
        for (int j = 0; j < FN; ++j) bf[j] = bs[(ks * 4 + lc) * LDB_S + j * 8];
#pragma unroll
        for (int i = 0; i < FM; ++i)
#pragma unroll
          for (int j = 0; j < FN; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
      }
    }
  }
  cp_async_wait<0>();

  // Epilogue: C fragment (row lr, cols 2*lc, 2*lc+1) straight to global through the index maps.
  double* out = p.out + (long long)blockIdx.z * p.split_stride;
#pragma unroll
  for (int i = 0; i < FM; ++i) {
    int r = m0 + wm0 + i * 8 + lr;
    if (r >= p.M) continue;
    long long roff = row_off[wm0 + i * 8 + lr];
#pragma unroll
    for (int j = 0; j < FN; ++j) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        int c = n0 + wn0 + j * 8 + 2 * lc + e;
        if (c < p.N) {
          long long off = roff + col_off[wn0 + j * 8 + 2 * lc + e];
          double v = acc[i][j][e];
          if (p.mode == 1) v = out[off] - v;
          else if (p.mode == 2) v = out[off] + v;
          out[off] = v;
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------
// Warp-specialised variant (the hot path for every large contraction, transA = 1):
//   * ONE producer warp stages the operands through the TMA engine, completion counted in bytes on the stage's
//     `full` mbarrier.  Default: one tiled bulk tensor copy per operand tile and k-step (cp.async.bulk.tensor.2d
//     through a tensor map, SASS UTMALDG, issued by one elected lane).  The box is BK rows of BM + PAD (BN + PAD)
//     columns - exactly the padded shared-memory pitch - so the dense box the copy engine writes is the padded,
//     bank-conflict-free layout (a BM-wide dense box would give 4-way conflicts on the 8-byte fragment loads and no
//     swizzle mode removes them); the PAD extra columns are the neighbour tile's and never read; ragged M / N / K
//     edges are zero-filled by the copy engine.  Batched launches and K-row maps (layered GEMM1): one linear bulk
//     copy (cp.async.bulk, SASS UBLKCP) per k-row of the A tile (lanes 0..15) and of the B tile (lanes 16..31),
//     widths clipped, missing k-rows of the last k-step zero-filled by the producer with ordinary stores.
//   * the consumer warps only do LDS.64 + DMMA and release a stage by arriving on its `empty` mbarrier -- no
//     CTA-wide barrier and no address arithmetic in the math warps (ncu history in profiles/r1_k4_gemm_ws_ncu.md:
//     cp.async kernel 71.6 % DMMA-active -> linear bulk copies 93.3 % -> tensor copies 96.4 %).
//   * SK = true: stream-K / hybrid schedules (GemmArgs::sk, sk_t1).
// Requires even leading dimensions and 16-byte aligned bases (checked on the host; otherwise the cp.async kernel
// above is used).
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
  asm volatile(
      "{\n.reg .pred p;\nWAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}\n" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void bulk_s2g(void* gdst, const void* ssrc, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n"
               ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;\n" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;\n" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* tm, int c0, int c1, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n"
               ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}

//   * RESB = true ("resident B", short-K GEMMs whose N fits one tile -- the two contractions of the layered absorption,
//     K = D^2 and d D^2): the whole K x N operand B is fetched ONCE per CTA into its own shared-memory region, the ring
//     streams only A tiles, and the CTAs are persistent (grid = resident CTA slots, work items dealt round robin), so
//     the producer warp prefetches the next tile's A rows while the consumers are still storing the previous tile.
template <int BM, int BN, int WM, int WN, int STAGES, bool SK = false, bool RESB = false>
__global__ void __launch_bounds__(((BM / WM) * (BN / WN) + 1) * 32, ((BM / WM) * (BN / WN) <= 4 ? 2 : 1))
gemm_f64_dmma_ws(const __grid_constant__ GemmArgs p) {
  constexpr int NW_M = BM / WM, NW_N = BN / WN, NCW = NW_M * NW_N;
  constexpr int LDA_S = BM + PAD, LDB_S = BN + PAD;
  constexpr int A_STAGE = BK * LDA_S, B_STAGE = BK * LDB_S;
  constexpr int FM = WM / 8, FN = WN / 8;
  static_assert(BK == 16, "one copy per lane: 16 A rows + 16 B rows");
  extern __shared__ __align__(128) double smem[];
  double* As = smem;
  double* Bs = smem + STAGES * A_STAGE;                 // RESB: all ceil(K / BK) k-tiles of B, else the ring's B stages
  const int nbst = RESB ? (p.K + BK - 1) / BK : STAGES;
  uint64_t* full = reinterpret_cast<uint64_t*>(Bs + nbst * B_STAGE);
  uint64_t* empty = full + STAGES;
  uint64_t* bfull = empty + STAGES;                     // RESB: B has landed (one phase per CTA)
  double* slabs = reinterpret_cast<double*>(empty + STAGES + 2);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // Persistent CTA: work items w = (z, tile_m, tile_n), tile_n fastest; the smem ring and its
  // mbarrier phases run on across work items, so the producer prefetches the next tile while the
  // consumers are still storing the previous one.
  const int tn = (p.N + BN - 1) / BN, tm = (p.M + BM - 1) / BM;
  const long long nwork = (long long)tn * tm * p.nz;
  const int nkt_total = (p.K + BK - 1) / BK;
  const long long w_begin = SK ? sk_first_unit(blockIdx.x, (long long)tn * tm * nkt_total, gridDim.x, p.sk_t1, nkt_total) : blockIdx.x;
  const long long w_end = SK ? sk_first_unit(blockIdx.x + 1, (long long)tn * tm * nkt_total, gridDim.x, p.sk_t1, nkt_total) : nwork;

  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, NCW); }
    mbar_init(bfull, 1);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  pdl_sync();

  if (warp == NCW) {
    // ------------------------------ producer warp
    const int row = lane & 15;
    const bool isB = lane >= 16;
    const int srow = isB ? row * LDB_S : row * LDA_S;
    int it = 0;                                   // k-tiles issued so far by this CTA (ring position)
    if (RESB && w_begin < w_end) {                // the whole B operand, once (N fits one tile: n0 = 0)
      int wBr = p.N < BN ? p.N : BN; wBr = (wBr + 1) & ~1;
      if (p.tma) {
        if (lane == 0) {
          mbar_expect_tx(bfull, (uint32_t)(nkt_total * BK * LDB_S) * 8u);
          for (int kt = 0; kt < nkt_total; ++kt) tma_load_2d(Bs + kt * B_STAGE, &p.tmB, 0, kt * BK, bfull);
        }
      } else {
        const int kz = (p.K + 3) & ~3;            // rows that complete the last k-step are zero-filled
        for (int kr = p.K + lane; kr < kz; kr += 32) {
          double* z = Bs + (kr / BK) * B_STAGE + (kr % BK) * LDB_S;
          for (int c = 0; c < BN; ++c) z[c] = 0.0;
        }
        __syncwarp();
        if (lane == 0) mbar_expect_tx(bfull, (uint32_t)p.K * (uint32_t)wBr * 8u);
        __syncwarp();
        for (int kr = lane; kr < p.K; kr += 32)
          bulk_g2s(Bs + (kr / BK) * B_STAGE + (kr % BK) * LDB_S, p.B + (long long)kr * p.ldb, (uint32_t)wBr * 8u, bfull);
      }
      __syncwarp();
    }
    for (long long w = w_begin; w < w_end;) {
      int z, rem, kt_begin, kt_end;
      if (SK) {
        z = 0; rem = (int)(w / nkt_total); kt_begin = (int)(w % nkt_total);
        const long long left = w_end - w;
        kt_end = left < nkt_total - kt_begin ? kt_begin + (int)left : nkt_total;
        w += kt_end - kt_begin;
      } else {
        z = (int)(w / ((long long)tn * tm)); rem = (int)(w % ((long long)tn * tm));
        kt_begin = p.batch ? 0 : z * p.ktiles_per_split;
        kt_end = kt_begin + p.ktiles_per_split; if (kt_end > nkt_total) kt_end = nkt_total;
        w += gridDim.x;
      }
      const int m0 = (rem / tn) * BM, n0 = (rem % tn) * BN;
      const double* Abase = p.A + (p.batch ? p.za(z) : 0);
      int wA = p.M - m0; if (wA > BM) wA = BM; wA = (wA + 1) & ~1;
      int wB = p.N - n0; if (wB > BN) wB = BN; wB = (wB + 1) & ~1;
      const uint32_t bytes = (uint32_t)(isB ? wB : wA) * 8u;
      if (p.tma) {
        for (int kt = kt_begin; kt < kt_end; ++kt, ++it) {
          const int stage = it % STAGES, round = it / STAGES;
          if (round > 0) mbar_wait(empty + stage, (round - 1) & 1);
          if (lane == 0) {
            mbar_expect_tx(full + stage, (uint32_t)(BK * (RESB ? LDA_S : LDA_S + LDB_S)) * 8u);
            tma_load_2d(As + stage * A_STAGE, &p.tmA, m0, kt * BK, full + stage);
            if (!RESB) tma_load_2d(Bs + stage * B_STAGE, &p.tmB, n0, kt * BK, full + stage);
          }
          __syncwarp();
        }
        continue;
      }
      for (int kt = kt_begin; kt < kt_end; ++kt, ++it) {
        const int stage = it % STAGES, round = it / STAGES;
        if (round > 0) mbar_wait(empty + stage, (round - 1) & 1);
        const int kr = kt * BK + row;                                 // logical k-row of this lane
        int krows = p.K - kt * BK; if (krows > BK) krows = BK;
        const double* src = isB ? p.B + (long long)kr * p.ldb + n0 : Abase + p.ka(kr) * p.lda + m0;
        double* dst = (isB ? Bs + (RESB ? 0 : stage) * B_STAGE : As + stage * A_STAGE) + srow;
        const bool mine = !(RESB && isB);                 // RESB: the B lanes have nothing to fetch per stage
        if (mine && row >= krows && row < ((krows + 3) & ~3)) {   // ragged K: zero the rows that complete the last k-step
          const int wz = isB ? BN : BM;                   // (the consumers stop after ceil(krows / 4) k-steps)
          for (int c = 0; c < wz; ++c) dst[c] = 0.0;
        }
        __syncwarp();
        if (lane == 0) mbar_expect_tx(full + stage, (uint32_t)krows * (uint32_t)(RESB ? wA : wA + wB) * 8u);
        __syncwarp();
        if (mine && row < krows) bulk_g2s(dst, src, bytes, full + stage);
      }
    }
    return;
  }

  // -------------------------------- consumer warps
  const int wm0 = (warp / NW_N) * WM, wn0 = (warp % NW_N) * WN;
  const int lr = lane >> 2, lc = lane & 3;
  int it = 0;
  if (RESB && w_begin < w_end) mbar_wait(bfull, 0);
  for (long long w = w_begin; w < w_end;) {
    int z, rem, kt_begin, kt_end;
    bool partial = false;
    int slot = 0;
    if (SK) {
      z = 0; rem = (int)(w / nkt_total); kt_begin = (int)(w % nkt_total);
      const long long left = w_end - w;
      kt_end = left < nkt_total - kt_begin ? kt_begin + (int)left : nkt_total;
      partial = kt_begin != 0 || kt_end != nkt_total;
      slot = 2 * ((int)blockIdx.x - p.sk_t1) + (w == w_begin ? 0 : 1);    // whole-tile CTAs never write a partial tile
      w += kt_end - kt_begin;
    } else {
      z = (int)(w / ((long long)tn * tm)); rem = (int)(w % ((long long)tn * tm));
      kt_begin = p.batch ? 0 : z * p.ktiles_per_split;
      kt_end = kt_begin + p.ktiles_per_split; if (kt_end > nkt_total) kt_end = nkt_total;
      w += gridDim.x;
    }
    const int m0 = (rem / tn) * BM, n0 = (rem % tn) * BN;

    // The output offsets of the tile's BM rows and BN columns (-1 = out of range) are worked out once per tile by
    // all consumer threads together, while the first operand tiles are still in flight, instead of up to 16
    // index-map evaluations (32 integer divisions) per thread after the main loop.
    long long* otab = reinterpret_cast<long long*>(slabs + NCW * 8 * (WN + 4));            // behind the staging slabs
    if (!(SK && partial)) {
      asm volatile("bar.sync 1, %0;\n" ::"n"(NCW * 32) : "memory");       // previous tile's epilogue has read the table
      for (int t = tid; t < BM + BN; t += NCW * 32) {
        const int g = t < BM ? m0 + t : n0 + t - BM;
        otab[t] = t < BM ? (g < p.M ? p.ro(g) : -1) : (g < p.N ? p.co(g) : -1);
      }
    }

    double acc[FM][FN][2];
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
      for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    for (int kt = kt_begin; kt < kt_end; ++kt, ++it) {
      const int stage = it % STAGES, round = it / STAGES;
      mbar_wait(full + stage, round & 1);
      const double* as = As + stage * A_STAGE + wm0 + lr + lc * LDA_S;
      const double* bs = Bs + (RESB ? kt : stage) * B_STAGE + wn0 + lr + lc * LDB_S;
      const int krows = p.K - kt * BK;
      if (krows >= BK) {
#pragma unroll
        for (int ks = 0; ks < BK / 4; ++ks) {
          double af[FM], bf[FN];
#pragma unroll
          for (int i = 0; i < FM; ++i) af[i] = as[ks * 4 * LDA_S + i * 8];
#pragma unroll
          for (int j = 0; j < FN; ++j) bf[j] = bs[ks * 4 * LDB_S + j * 8];
#pragma unroll
          for (int i = 0; i < FM; ++i)
#pragma unroll
            for (int j = 0; j < FN; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
      } else {
        const int ksteps = (krows + 3) >> 2;
        for (int ks = 0; ks < ksteps; ++ks) {
          double af[FM], bf[FN];
#pragma unroll
          for (int i = 0; i < FM; ++i) af[i] = as[ks * 4 * LDA_S + i * 8];
#pragma unroll
          for (int j = 0; j < FN; ++j) bf[j] = bs[ks * 4 * LDB_S + j * 8];
#pragma unroll
          for (int i = 0; i < FM; ++i)
#pragma unroll
            for (int j = 0; j < FN; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty + stage);
    }

    double* out = p.out + (p.batch ? (long long)z * p.zo : (long long)z * p.split_stride);
    if (SK && partial) {
      // stream-K partial tile: plain BM x BN slab, no maps, no bounds (the fix-up reads the valid part only)
      double* slab = p.sk_ws + (long long)slot * (BM * BN) + (wm0 + lr) * BN + wn0 + 2 * lc;
#pragma unroll
      for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < FN; ++j)
          *reinterpret_cast<double2*>(slab + i * 8 * BN + j * 8) = make_double2(acc[i][j][0], acc[i][j][1]);
    } else if (p.epi == 2) {
      // dense blocks: slab layout [group][8 rows][wc]; lane g stores group g's block (split where the rows of the
      // block are not consecutive in the output: a row-map boundary, or the ragged end of M)
      const int wc = p.dense_wc, magic = p.dense_magic;
      double* stg = slabs + warp * (8 * (WN + 4));
      const int ng = (p.N - wn0 < WN ? p.N - wn0 : WN) / wc;          // column groups of this warp
      asm volatile("bar.sync 1, %0;\n" ::"n"(NCW * 32) : "memory");       // offset table complete
#pragma unroll
      for (int i = 0; i < FM; ++i) {
        if (lane < ng) bulk_wait_read0();                               // the slab's previous block has been read
        __syncwarp();
#pragma unroll
        for (int j = 0; j < FN; ++j) {
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const int c = j * 8 + 2 * lc + e;
            const int g = (c * magic) >> 16;
            if (g < ng) stg[(g * 8 + lr) * wc + (c - g * wc)] = acc[i][j][e];
          }
        }
        fence_async_smem();
        __syncwarp();
        if (lane < ng) {
          const long long cgo = otab[BM + wn0 + lane * wc];
          const long long* rt = otab + wm0 + i * 8;
          const double* src = stg + lane * 8 * wc;
          int rr = 0;
          while (rr < 8) {
            const long long o0 = rt[rr];
            if (o0 < 0) break;                                          // rows beyond M sit at the end of the tile
            int len = 1;
            while (rr + len < 8 && rt[rr + len] == o0 + (long long)len * wc) ++len;
            bulk_s2g(out + o0 + cgo, src + rr * wc, (uint32_t)(len * wc) * 8u);
            rr += len;
          }
          bulk_commit();
        }
      }
      if (lane < ng) bulk_wait_read0();
      __syncwarp();
    } else if (p.epi == 1) {
      // staged: 8 rows x WN columns of this warp go through its private shared-memory slab, then every
      // store instruction writes 32 consecutive columns of one row (coalesced wherever co() is contiguous)
      constexpr int SP = WN + 4, NCH = (WN + 31) / 32;
      double* stg = slabs + warp * (8 * SP);
      asm volatile("bar.sync 1, %0;\n" ::"n"(NCW * 32) : "memory");       // offset table complete
      long long coffL[NCH];
#pragma unroll
      for (int q = 0; q < NCH; ++q) {
        const int cl = q * 32 + lane;
        coffL[q] = cl < WN ? otab[BM + wn0 + cl] : -1;
      }
#pragma unroll
      for (int i = 0; i < FM; ++i) {
        const long long myro = lane < 8 ? otab[wm0 + i * 8 + lane] : -1;
#pragma unroll
        for (int j = 0; j < FN; ++j) {
          double2 v2 = make_double2(acc[i][j][0], acc[i][j][1]);
          *reinterpret_cast<double2*>(stg + lr * SP + j * 8 + 2 * lc) = v2;
        }
        __syncwarp();
#pragma unroll
        for (int rr = 0; rr < 8; ++rr) {
          const long long roff = __shfl_sync(0xffffffffu, myro, rr);
          if (roff < 0) continue;
#pragma unroll
          for (int q = 0; q < NCH; ++q) {
            if (coffL[q] >= 0) {
              const long long off = roff + coffL[q];
              double v = stg[rr * SP + q * 32 + lane];
              if (p.mode == 1) v = out[off] - v;
              else if (p.mode == 2) v = out[off] + v;
              out[off] = v;
            }
          }
        }
        __syncwarp();
      }
    } else {
      asm volatile("bar.sync 1, %0;\n" ::"n"(NCW * 32) : "memory");       // offset table complete
      long long coff[FN][2];
#pragma unroll
      for (int j = 0; j < FN; ++j) {
        const longlong2 c2 = *reinterpret_cast<const longlong2*>(otab + BM + wn0 + j * 8 + 2 * lc);
        coff[j][0] = c2.x; coff[j][1] = c2.y;
      }
      if (p.mode == 0) {
#pragma unroll
        for (int i = 0; i < FM; ++i) {
          const long long roff = otab[wm0 + i * 8 + lr];
          if (roff < 0) continue;
          double* orow = out + roff;
#pragma unroll
          for (int j = 0; j < FN; ++j) {
            if (coff[j][0] >= 0) orow[coff[j][0]] = acc[i][j][0];
            if (coff[j][1] >= 0) orow[coff[j][1]] = acc[i][j][1];
          }
        }
      } else {
        const double sgn = p.mode == 1 ? -1.0 : 1.0;
#pragma unroll
        for (int i = 0; i < FM; ++i) {
          const long long roff = otab[wm0 + i * 8 + lr];
          if (roff < 0) continue;
          double* orow = out + roff;
#pragma unroll
          for (int j = 0; j < FN; ++j) {
#pragma unroll
            for (int e = 0; e < 2; ++e)
              if (coff[j][e] >= 0) orow[coff[j][e]] = fma(sgn, acc[i][j][e], orow[coff[j][e]]);
          }
        }
      }
    }
  }
  if (p.epi == 2) bulk_wait0();                   // every bulk store of this thread has completed
}

// Plain DFMA reference kernel (QRCTM_OPT_GEMM_PATH = 1): one output element per
// thread, no tiling.  Only for debugging / cross-checking the DMMA path on the GPU.
__global__ void gemm_f64_ref(GemmArgs p) {
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)p.M * p.N) return;
  int i = (int)(idx / p.N), j = (int)(idx % p.N);
  const double* A = p.A + (p.batch ? p.za((int)blockIdx.z) : 0);
  double* out = p.out + (p.batch ? (long long)blockIdx.z * p.zo : 0);
  double s = 0.0;
  for (int k = 0; k < p.K; ++k) {
    double a = p.transA ? A[p.ka(k) * p.lda + i] : A[(long long)i * p.lda + k];
    s = fma(a, p.B[(long long)k * p.ldb + j], s);
  }
  long long off = p.ro(i) + p.co(j);
  if (p.mode == 1) s = out[off] - s;
  else if (p.mode == 2) s = out[off] + s;
  out[off] = s;
}

// out[ro(i)+co(j)] (op)= sum_z part[z][i][j], z ascending (fixed order).
__global__ void reduce_splitk(const double* part, long long split_stride, int splits, int M, int N,
                              double* out, IndexMap ro, IndexMap co, int mode) {
  pdl_sync();
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)M * N) return;
  int i = (int)(idx / N), j = (int)(idx % N);
  double s = 0.0;
  int z = 0;
  for (; z + 8 <= splits; z += 8) {            // 8 loads in flight, summed in ascending z (fixed order)
    double v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = part[(long long)(z + u) * split_stride + idx];
#pragma unroll
    for (int u = 0; u < 8; ++u) s += v[u];
  }
  for (; z < splits; ++z) s += part[(long long)z * split_stride + idx];
  long long off = ro(i) + co(j);
  if (mode == 1) s = out[off] - s;
  else if (mode == 2) s = out[off] + s;
  out[off] = s;
}

// Stream-K fix-up: gridDim.x = output tiles, gridDim.y = row slices of a tile.  The CTAs that hold a part of tile t's
// k range are found from the same arithmetic the GEMM used (thread 0, once per CTA); if one of them covered the whole
// range the tile was stored directly and nothing is done.
// out[ro(i)+co(j)] (op)= sum of the partial tiles in ascending k (= ascending CTA index: fixed order).
constexpr int SK_MAXSEG = 320;
__global__ void __launch_bounds__(256)
streamk_fixup(const double* __restrict__ ws, int BM, int BN, int tn, int nkt, long long units, int ncta, int t1, int M,
              int N, double* out, IndexMap ro, IndexMap co, int mode) {
  __shared__ int slots[SK_MAXSEG];
  __shared__ int nseg_s;
  pdl_sync();
  const int t = t1 + blockIdx.x;                             // tiles below t1 were stored directly
  if (threadIdx.x == 0) {
    const long long ub = (long long)t * nkt, ue = ub + nkt;
    long long c = t1 + (ub - (long long)t1 * nkt) * (ncta - t1) / (units - (long long)t1 * nkt);
    while (c + 1 < ncta && sk_first_unit(c + 1, units, ncta, t1, nkt) <= ub) ++c;
    while (c > t1 && sk_first_unit(c, units, ncta, t1, nkt) > ub) --c;
    int nseg = 0;
    for (; c < ncta && nseg < SK_MAXSEG; ++c) {
      const long long u0 = sk_first_unit(c, units, ncta, t1, nkt), u1 = sk_first_unit(c + 1, units, ncta, t1, nkt);
      if (u0 >= ue) break;
      if (u0 <= ub && u1 >= ue) { nseg = 0; break; }         // whole tile by one CTA: stored directly
      if (u1 > u0) slots[nseg++] = (int)(2 * (c - t1) + (u0 >= ub ? 0 : 1));   // first segment of CTA c, else its last
    }
    nseg_s = nseg;
  }
  __syncthreads();
  const int nseg = nseg_s;
  if (nseg == 0) return;
  const int m0 = (t / tn) * BM, n0 = (t % tn) * BN;
  const int hrows = M - m0 < BM ? M - m0 : BM, wcols = N - n0 < BN ? N - n0 : BN;
  const long long tile = (long long)BM * BN;
  const int rows_per = (hrows + gridDim.y - 1) / gridDim.y;
  const int i0 = blockIdx.y * rows_per, i1 = i0 + rows_per < hrows ? i0 + rows_per : hrows;
  for (int i = i0 + threadIdx.x / 32; i < i1; i += blockDim.x / 32) {
    const long long roff = ro(m0 + i);
    for (int j = threadIdx.x % 32; j < wcols; j += 32) {
      const double* src = ws + (long long)i * BN + j;
      double s = 0.0;
      int q = 0;
      for (; q + 4 <= nseg; q += 4) {
        const double v0 = src[slots[q] * tile], v1 = src[slots[q + 1] * tile], v2 = src[slots[q + 2] * tile],
                     v3 = src[slots[q + 3] * tile];
        s += v0; s += v1; s += v2; s += v3;
      }
      for (; q < nseg; ++q) s += src[slots[q] * tile];
      const long long off = roff + co(n0 + j);
      if (mode == 1) s = out[off] - s;
      else if (mode == 2) s = out[off] + s;
      out[off] = s;
    }
  }
}

}  // namespace qk
