// libqrctm.so -- C ABI (include/qrctm.h) and the iteration driver (K9).
// Links only cudart.  No cuBLAS / cuSOLVER / libtorch.
#include "../../include/qrctm.h"

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "gemm_f64.cuh"
#include "kernels_misc.cuh"
#include "qr_f64.cuh"
#include "spectrum.cuh"
#include "eigh.cuh"

using namespace qk;

namespace {

constexpr int kPartialBlocks = 592;   // 4 x 148 blocks for the reduction kernels
constexpr size_t kAlign = 256;

inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct Layout {   // byte offsets into the workspace
  size_t A, a_mat, a2_mat, LH, rho, B1, B2, P1, C, T, Cn, Tn, X, Q, R, Rt, P, S, W, E, splitk, partial, scal, flag, Wc, dvec, evec,
      vv, pv, eig, s, s_prev, s_tmp, delta, qrwork, total;
  long long lda_a, ld1, ld2;
  size_t splitk_elems, qrwork_bytes;
};

}  // namespace

struct qrctm {
  int d, D, b, chi;       // chi: current bond dimension (<= chi_cap; below it only during the NEXT-2 warm-up)
  int chi_cap;            // the chi the workspace was sized for
  long long m;            // chi * b
  int eig_rows, eig_cols; // shape of U left in Q by the last eigen step (0: none)
  void* eigwork;          // NEXT-2 eigensolver workspace, allocated by the first qrctm_eig_step
  size_t eigwork_bytes;
  cudaStream_t stream;
  char* base;             // workspace
  bool owns_ws;
  Layout L;
  bool have_A, have_env;
  int corner_mode, symmetrize, check_every, gemm_path, time_stages, qr_path, absorb_mode;
  long long launches;
  cudaEvent_t ev[QRCTM_NSTAGE + 2];
  bool have_ev;
  cudaGraphExec_t g_front, g_k7;  // captured K1..K6 and K7 (replayed by step/run)
  long long g_front_n, g_k7_n;    // kernels per replay
  int use_graph, warm_steps, graph_failed;
  int need_s0;                    // spectrum of the environment set by set_env not computed yet (lazy)
  cudaStream_t side;            // high-priority stream for the overlapped convergence check
  cudaEvent_t ev_env, ev_spec;  // environment ready (main) / spectrum done (side)
  int overlap;
  double stage_ms[QRCTM_NSTAGE + 1];
  long long stage_steps;
  char err[256];
  double* h_pinned;       // [0] delta, [1..] scratch ; pinned host
  int* h_flag;
  // typed views
  double *A, *a_mat, *a2_mat, *LH, *rho, *B1, *B2, *P1, *C, *T, *Cn, *Tn, *X, *Q, *R, *Rt, *P, *S, *W, *E, *splitk, *partial, *scal, *Wc,
      *dvec, *evec, *vv, *pv, *eig, *s, *s_prev, *s_tmp, *delta;
  int* flag;
  void* qrwork;
};

namespace {

unsigned long long qr_work_bytes_impl(long long rows, int cols);

bool make_layout(int d, int D, int chi, Layout* L) {
  if (d < 1 || D < 1 || chi < 1) return false;
  if (D > 32 || chi > 1024 || d > 64) return false;                  // sizes this build supports
  long long b = (long long)D * D, m = b * chi;
  long long b2 = b * b;
  L->lda_a = (b2 + 15) / 16 * 16;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
  const size_t dbl = sizeof(double);
  L->A = take(dbl * d * b2);
  L->a_mat = take(dbl * b2 * L->lda_a);
  L->a2_mat = take(dbl * b2 * L->lda_a);
  L->LH = take(d <= 4 ? dbl * (size_t)d * d * m * chi : 0);
  L->rho = take(dbl * 256);
  L->ld1 = ((long long)d * b + 15) / 16 * 16;
  L->ld2 = (b + 15) / 16 * 16;
  L->B1 = take(dbl * b * L->ld1);
  L->B2 = take(dbl * d * b * L->ld2);
  L->P1 = take(dbl * (size_t)d * b * (size_t)chi * chi * b);
  L->C = take(dbl * chi * chi);
  L->T = take(dbl * m * chi);
  L->Cn = take(dbl * chi * chi);
  L->Tn = take(dbl * m * chi);
  L->X = take(dbl * m * chi);
  L->Q = take(dbl * m * chi);
  L->R = take(dbl * chi * chi);
  L->Rt = take(dbl * chi * chi);
  L->P = take(dbl * m * m);
  L->S = take(dbl * m * m);
  L->W = take(dbl * m * chi);
  L->E = take(dbl * m * chi);
  L->splitk_elems = (size_t)256 * chi * chi + (size_t)16 * m * chi;
  L->splitk = take(dbl * L->splitk_elems);
  L->partial = take(dbl * 4 * kPartialBlocks);
  L->scal = take(dbl * 16);
  L->flag = take(sizeof(int) * 4);
  L->Wc = take(dbl * chi * chi);
  L->dvec = take(dbl * chi);
  L->evec = take(dbl * chi);
  L->vv = take(dbl * chi);
  L->pv = take(dbl * chi);
  L->eig = take(dbl * chi);
  L->s = take(dbl * chi);
  L->s_prev = take(dbl * chi);
  L->s_tmp = take(dbl * chi);
  L->delta = take(dbl * 4);
  L->qrwork_bytes = qr_work_bytes_impl(m, chi);
  L->qrwork = take(L->qrwork_bytes);
  L->total = off;
  return true;
}

void bind_views(qrctm* h) {
  char* B = h->base;
  const Layout& L = h->L;
#define V_(name) h->name = reinterpret_cast<double*>(B + L.name)
  V_(A); V_(a_mat); V_(a2_mat); V_(LH); V_(rho); V_(B1); V_(B2); V_(P1); V_(C); V_(T); V_(Cn); V_(Tn); V_(X); V_(Q); V_(R); V_(Rt); V_(P); V_(S); V_(W);
  V_(E); V_(splitk); V_(partial); V_(scal); V_(Wc); V_(dvec); V_(evec); V_(vv); V_(pv); V_(eig); V_(s);
  V_(s_prev); V_(s_tmp); V_(delta);
#undef V_
  h->flag = reinterpret_cast<int*>(B + L.flag);
  h->qrwork = B + L.qrwork;
}

int fail(qrctm* h, int code, const char* what, cudaError_t e = cudaSuccess) {
  if (h) {
    if (e != cudaSuccess) snprintf(h->err, sizeof(h->err), "%s: %s", what, cudaGetErrorString(e));
    else snprintf(h->err, sizeof(h->err), "%s", what);
  }
  return code;
}

#define CU(h, call)                                                        \
  do {                                                                     \
    cudaError_t e__ = (call);                                              \
    if (e__ != cudaSuccess) return fail((h), QRCTM_ERR_CUDA, #call, e__);  \
  } while (0)

bool is_device_ptr(const void* p) {
  cudaPointerAttributes at;
  cudaError_t e = cudaPointerGetAttributes(&at, p);
  if (e != cudaSuccess) { cudaGetLastError(); return false; }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

cudaError_t copy_in(double* dst_dev, const double* src, size_t n, cudaStream_t st) {
  cudaMemcpyKind k = is_device_ptr(src) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  cudaError_t e = cudaMemcpyAsync(dst_dev, src, n * sizeof(double), k, st);
  if (e != cudaSuccess) return e;
  return k == cudaMemcpyHostToDevice ? cudaStreamSynchronize(st) : cudaSuccess;
}
cudaError_t copy_out(double* dst, const double* src_dev, size_t n, cudaStream_t st) {
  cudaMemcpyKind k = is_device_ptr(dst) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  cudaError_t e = cudaMemcpyAsync(dst, src_dev, n * sizeof(double), k, st);
  if (e != cudaSuccess) return e;
  return cudaStreamSynchronize(st);
}

// ------------------------------------------------------------------ GEMM launcher
template <int BM, int BN, int WM, int WN, int STAGES>
cudaError_t launch_cfg(cudaStream_t st, const GemmArgs& g, int splits) {
  constexpr int NT = (BM / WM) * (BN / WN) * 32;
  constexpr size_t smem = sizeof(double) * STAGES * BK * ((BM + PAD) + (BN + PAD));
  static bool attr_done = false;
  if (!attr_done) {
    cudaError_t e = cudaFuncSetAttribute(gemm_f64_dmma<BM, BN, WM, WN, STAGES>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_done = true;
  }
  dim3 grid((g.N + BN - 1) / BN, (g.M + BM - 1) / BM, splits);
  gemm_f64_dmma<BM, BN, WM, WN, STAGES><<<grid, NT, smem, st>>>(g);
  return cudaGetLastError();
}

template <int BM, int BN, int WM, int WN, int STAGES>
cudaError_t launch_cfg_ws(cudaStream_t st, const GemmArgs& g, int splits) {
  constexpr int NT = ((BM / WM) * (BN / WN) + 1) * 32;
  constexpr size_t smem = sizeof(double) * STAGES * BK * ((BM + PAD) + (BN + PAD)) + 2 * STAGES * sizeof(uint64_t) +
                          sizeof(double) * (BM / WM) * (BN / WN) * 8 * (WN + 4);     // + per-warp epilogue slabs
  static bool attr_done = false;
  if (!attr_done) {
    cudaError_t e = cudaFuncSetAttribute(gemm_f64_dmma_ws<BM, BN, WM, WN, STAGES>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_done = true;
  }
  static int nslots = 0;
  if (!nslots) {
    int dev = 0, nsm = 148, per = 1;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, gemm_f64_dmma_ws<BM, BN, WM, WN, STAGES>, NT, smem);
    nslots = nsm * (per > 0 ? per : 1);
  }
  GemmArgs ga = g;
  ga.nz = splits;
  const long long nwork = (long long)((g.N + BN - 1) / BN) * ((g.M + BM - 1) / BM) * splits;
  (void)nslots;                                  // one work item per CTA: the hardware scheduler balances better
  const unsigned grid = (unsigned)nwork;         // than a static persistent loop (measured)
  gemm_f64_dmma_ws<BM, BN, WM, WN, STAGES><<<grid, NT, smem, st>>>(ga);
  return cudaGetLastError();
}

struct GemmCall {
  const double* A; long long lda; int transA;
  const double* B; long long ldb;
  double* out; IndexMap ro, co;
  int M, N, K;
  int mode;   // 0 store, 1 out -= , 2 out +=
  IndexMap ka = IndexMap{1, 1, 0};     // k-row map of A (transA = 1)
  int batch = 0;                       // > 0: gridDim.z batches, A += za(z), out += z * zo
  IndexMap za = IndexMap{1, 0, 0};
  long long zo = 0;
  int epi = 0;                         // 1: shared-memory staged epilogue (outputs contiguous along the column index)
};

// Returns number of kernels launched (>0) or -1 on error (err set).
int launch_gemm(cudaStream_t st, int path, const GemmCall& c, double* splitk_ws, size_t splitk_elems,
                cudaError_t* err) {
  *err = cudaSuccess;
  if (c.M <= 0 || c.N <= 0) return 0;
  GemmArgs g;
  g.A = c.A; g.lda = c.lda; g.transA = c.transA; g.B = c.B; g.ldb = c.ldb; g.out = c.out;
  g.ro = c.ro; g.co = c.co; g.M = c.M; g.N = c.N; g.K = c.K; g.mode = c.mode;
  g.ka = c.ka; g.batch = c.batch > 0 ? 1 : 0; g.za = c.za; g.zo = c.zo; g.epi = c.epi;
  g.vecA = c.transA && (c.lda % 2 == 0) && ((reinterpret_cast<uintptr_t>(c.A) & 15) == 0);
  g.vecB = (c.ldb % 2 == 0) && ((reinterpret_cast<uintptr_t>(c.B) & 15) == 0);
  g.split_stride = 0;
  const int nkt = (c.K + BK - 1) / BK;
  g.ktiles_per_split = nkt > 0 ? nkt : 1;
  if (path == 1) {
    long long n = (long long)c.M * c.N;
    gemm_f64_ref<<<dim3((unsigned)((n + 255) / 256), 1, c.batch > 0 ? c.batch : 1), 256, 0, st>>>(g);
    *err = cudaGetLastError();
    return *err == cudaSuccess ? 1 : -1;
  }
  const long long t128 = (long long)((c.M + 127) / 128) * ((c.N + 127) / 128);
  const long long t64 = (long long)((c.M + 63) / 64) * ((c.N + 63) / 64);
  const bool big = t128 >= 120;
  const bool ws_ok = g.transA && g.vecA && g.vecB;     // bulk copies need 16-byte aligned rows
  int splits = 1;
  int cfg = 0;          // 0: 64x64 cp.async, 1: 128x128 cp.async, 2: ws 128x128, 3: ws 128x104, 4: ws 128x64 (2 CTA/SM)
  const bool ws_big = ws_ok && c.M >= 96 && c.N >= 32 && (double)c.M * c.N * c.K > 2.0e8;
  if (c.batch > 0) {
    // batched launch (layered absorption): bulk-copy kernel only, one batch per gridDim.z, no split-K
    if (!ws_ok) { *err = cudaErrorInvalidValue; return -1; }
    const int pad128 = (c.N + 127) / 128 * 128, pad104 = (c.N + 103) / 104 * 104, pad64 = (c.N + 63) / 64 * 64;
    if (c.N <= 56) *err = launch_cfg_ws<128, 56, 32, 56, 3>(st, g, c.batch);
    else if (pad64 <= pad104 && pad64 <= pad128) *err = launch_cfg_ws<128, 64, 64, 32, 4>(st, g, c.batch);
    else if (pad104 <= pad128 && nkt <= 6) *err = launch_cfg_ws<64, 104, 16, 104, 3>(st, g, c.batch);   // 2 CTAs/SM
    else if (pad104 <= pad128) *err = launch_cfg_ws<128, 104, 16, 104, 4>(st, g, c.batch);
    else *err = launch_cfg_ws<128, 128, 64, 32, 4>(st, g, c.batch);
    return *err == cudaSuccess ? 1 : -1;
  }
  if (ws_big) {
    // pick the N tile with the least padding, then split K so that the CTAs fill whole waves
    auto padded = [&](int bn) { return (long long)((c.N + bn - 1) / bn) * bn; };
    int bn = 128; cfg = 2;
    if (c.N <= 56) { bn = 56; cfg = 5; }                       // narrow N (layered absorption, N = D^2)
    else if (c.N <= 64) { bn = 64; cfg = 4; }
    else if (c.N >= 1024) { bn = 64; cfg = 4; }                // wide N: two CTAs per SM overlap epilogue and main loop
                                                               // (K4 at cfg4: 13.10 ms vs 13.20 ms with 128x128, 13.20 with 128x56)
    else if (padded(104) * 100 < padded(128) * 97) { bn = 104; cfg = 3; }
    const long long tiles = (long long)((c.M + 127) / 128) * ((c.N + bn - 1) / bn);
    const int slots = (cfg == 4 || cfg == 5) ? 296 : 148;
    const double t_kt = 2.1e-6 * bn / 128.0 * ((cfg == 4 || cfg == 5) ? 2.0 : 1.0), t_fix = 4e-6;
    double best = 1e30;
    for (int sp = 1; sp <= 64; ++sp) {
      int per = (nkt + sp - 1) / sp;
      if (sp > 1 && per < 8) break;
      int sp_eff = (nkt + per - 1) / per;
      if (sp_eff != sp) continue;
      if (sp > 1 && (size_t)c.M * c.N * sp > splitk_elems) break;
      long long waves = (tiles * sp + slots - 1) / slots;
      double t = waves * (per * t_kt + t_fix) + (sp > 1 ? 2.0 * sp * c.M * (double)c.N * 8.0 / 4e12 + 4e-6 : 0.0);
      if (t < best * 0.97) { best = t; splits = sp; }
    }
  } else if (big) {
    cfg = 1;
  } else if (t64 < 148 && nkt >= 8) {
    splits = (int)((2 * 148 + t64 - 1) / t64);
    if (splits > nkt / 2) splits = nkt / 2;
    size_t per = (size_t)c.M * c.N;
    if (per * splits > splitk_elems) splits = (int)(splitk_elems / per);
    if (splits < 1) splits = 1;
  }
  int launched = 0;
  if (splits > 1) {
    g.ktiles_per_split = (nkt + splits - 1) / splits;
    splits = (nkt + g.ktiles_per_split - 1) / g.ktiles_per_split;
    g.out = splitk_ws; g.ro = plain_map(c.N); g.co = IndexMap{1, 1, 0}; g.mode = 0;
    g.split_stride = (long long)c.M * c.N;
  }
  switch (cfg) {
    case 2: *err = launch_cfg_ws<128, 128, 64, 32, 4>(st, g, splits); break;
    case 3: *err = launch_cfg_ws<128, 104, 16, 104, 4>(st, g, splits); break;
    case 4: *err = launch_cfg_ws<128, 64, 64, 32, 4>(st, g, splits); break;
    case 5: *err = launch_cfg_ws<128, 56, 32, 56, 3>(st, g, splits); break;
    case 1: *err = launch_cfg<128, 128, 64, 32, 4>(st, g, splits); break;
    default: *err = launch_cfg<64, 64, 32, 32, 4>(st, g, splits); break;
  }
  if (*err != cudaSuccess) return -1;
  ++launched;
  if (splits > 1) {
    long long n = (long long)c.M * c.N;
    reduce_splitk<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(splitk_ws, g.split_stride, splits, c.M, c.N,
                                                              c.out, c.ro, c.co, c.mode);
    *err = cudaGetLastError();
    if (*err != cudaSuccess) return -1;
    ++launched;
  }
  return launched;
}

}  // namespace

// ------------------------------------------------------------------ K2: QR driver
namespace {

constexpr int QR_NB = 16;        // shared-memory / global panel kernel (fallback for very tall panels)
constexpr int QR_NB_REG = 16;    // register-resident panel kernel (default)
constexpr int QR_REG_NT = 256, QR_REG_RPT = 40;                       // 640 rows per CTA
constexpr int QR_MAX_PARTS = 320;

struct QrWork {     // carved out of the caller's work buffer
  double *V, *Vc, *tau, *Tfac, *W1, *W2, *splitk, *part, *Vct, *Gq, *Xq;
  size_t splitk_elems;
};

size_t qr_layout(long long rows, int n, char* base, QrWork* w) {
  size_t off = 0;
  auto take = [&](size_t elems) { size_t o = off; off = align_up(off + sizeof(double) * elems); return o; };
  size_t oV = take((size_t)rows * n), oVc = take((size_t)rows * n), otau = take(n);
  size_t npan = (n + QR_NB - 1) / QR_NB;
  size_t oT = take(npan * QR_NB_REG * QR_NB_REG), oW1 = take((size_t)QR_NB_REG * n), oW2 = take((size_t)QR_NB_REG * n);
  size_t sk = (size_t)512 * QR_NB * n;
  size_t oS = take(sk);
  size_t oP = take((size_t)QR_MAX_PARTS * QR_NB_REG * n);
  size_t oVt = take((size_t)rows * n), oG = take((size_t)n * n), oX = take((size_t)n * n);
  if (w) {
    w->V = reinterpret_cast<double*>(base + oV); w->Vc = reinterpret_cast<double*>(base + oVc);
    w->tau = reinterpret_cast<double*>(base + otau); w->Tfac = reinterpret_cast<double*>(base + oT);
    w->W1 = reinterpret_cast<double*>(base + oW1); w->W2 = reinterpret_cast<double*>(base + oW2);
    w->splitk = reinterpret_cast<double*>(base + oS); w->splitk_elems = sk;
    w->part = reinterpret_cast<double*>(base + oP);
    w->Vct = reinterpret_cast<double*>(base + oVt); w->Gq = reinterpret_cast<double*>(base + oG);
    w->Xq = reinterpret_cast<double*>(base + oX);
  }
  return off;
}

unsigned long long qr_work_bytes_impl(long long rows, int cols) {
  if (rows < 1 || cols < 1) return 0;
  return qr_layout(rows, cols, nullptr, nullptr);
}

// X (rows x n, ld n, DEVICE, untouched) -> Q (rows x n), R (n x n), diag(R) >= 0.
// Level-2 Householder (one reflector at a time).  Returns kernels launched or -1.
long long qr_factor_level2(cudaStream_t st, long long rows, int n, const double* X, double* Q, double* R,
                           void* work, cudaError_t* err) {
  QrWork wk;
  qr_layout(rows, n, static_cast<char*>(work), &wk);
  double* V = wk.V;
  double* tau = wk.tau;
  long long launches = 0;
  *err = cudaMemcpyAsync(V, X, sizeof(double) * rows * n, cudaMemcpyDeviceToDevice, st);
  if (*err != cudaSuccess) return -1;
  constexpr int CPB = 4;
  for (int k = 0; k < n; ++k) {
    house_col_kernel<<<1, 1024, 0, st>>>(V, n, rows, k, tau);
    ++launches;
    if (k + 1 < n) {
      int nb = (n - (k + 1) + CPB - 1) / CPB;
      house_apply_kernel<CPB><<<nb, 512, 0, st>>>(V, n, rows, k, tau, V, n, k + 1, n);
      ++launches;
    }
  }
  copy_triu_kernel<<<(n * n + 255) / 256, 256, 0, st>>>(V, n, n, R);
  set_identity_top_kernel<<<296, 256, 0, st>>>(Q, rows, n);
  launches += 2;
  for (int k = n - 1; k >= 0; --k) {
    int nb = (n - k + CPB - 1) / CPB;
    house_apply_kernel<CPB><<<nb, 512, 0, st>>>(V, n, rows, k, tau, Q, n, k, n);
    ++launches;
  }
  sign_fix_kernel<<<296, 256, 0, st>>>(Q, rows, n, R);
  sign_fix_R_kernel<<<n, 128, 0, st>>>(R, n);
  launches += 2;
  *err = cudaGetLastError();
  return *err == cudaSuccess ? launches : -1;
}

// Panel launch: one cluster of C CTAs x 1024 threads.
cudaError_t launch_panel(cudaStream_t st, double* V, long long ld, long long m, int j0, int nbw, double* Vc,
                         double* tau, double* Tp) {
  constexpr int NB = QR_NB;
  static int max_smem = -1, cluster16 = -1;
  if (max_smem < 0) {
    int dev = 0; cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaError_t e = cudaFuncSetAttribute(qr_panel_cluster_kernel<NB, true>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(qr_panel_cluster_kernel<NB, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             max_smem);
    if (e != cudaSuccess) return e;
    cluster16 = (cudaFuncSetAttribute(qr_panel_cluster_kernel<NB, true>,
                                      cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess &&
                 cudaFuncSetAttribute(qr_panel_cluster_kernel<NB, false>,
                                      cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) ? 1 : 0;
    cudaGetLastError();
  }
  const long long prow = m - j0;
  constexpr int NP = NB * NB, NQ = 1024 / NP > 0 ? 1024 / NP : 1;
  const size_t fixed = sizeof(double) * (2 * 16 * NB + 2 * NB + 32 * NB + 3 * NB + (NB + 2) + NP + 16 * NP + NQ * NP);
  int C = 8;
  if (prow < 8 * 64) C = prow >= 256 ? 4 : (prow >= 64 ? 2 : 1);
  long long rpc = (prow + C - 1) / C;
  size_t slice = sizeof(double) * (size_t)rpc * NB;
  bool use_smem = true;
  if (fixed + slice > (size_t)max_smem) {
    if (cluster16) { C = 16; rpc = (prow + C - 1) / C; slice = sizeof(double) * (size_t)rpc * NB; }
    if (fixed + slice > (size_t)max_smem) { use_smem = false; slice = 0; }
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(C); cfg.blockDim = dim3(1024);
  cfg.dynamicSmemBytes = fixed + slice; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return use_smem ? cudaLaunchKernelEx(&cfg, qr_panel_cluster_kernel<NB, true>, V, ld, m, j0, nbw, Vc, tau, Tp, rpc)
                  : cudaLaunchKernelEx(&cfg, qr_panel_cluster_kernel<NB, false>, V, ld, m, j0, nbw, Vc, tau, Tp, rpc);
}

// Register-resident panel launch.  Returns cudaErrorInvalidValue if the panel is too tall for it.
int reg_panel_max_cluster() {
  static int maxc = -1;
  if (maxc < 0) {
    auto k = qr_panel_reg2_kernel<QR_NB_REG, QR_REG_NT, QR_REG_RPT, true>;
    maxc = cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess ? 16 : 8;
    cudaGetLastError();
  }
  return maxc;
}

cudaError_t launch_panel_reg(cudaStream_t st, double* V, long long ld, long long m, int j0, int nbw, double* Vc,
                             double* tau, double* Tp) {
  constexpr int cap = QR_REG_RPT * (QR_REG_NT / QR_NB_REG);
  const long long prow = m - j0;
  const int maxc = reg_panel_max_cluster();
  int C = 1;
  while (C < maxc && (prow + C - 1) / C > cap) C *= 2;
  const long long rpc = (prow + C - 1) / C;
  if (rpc > cap) return cudaErrorInvalidValue;
  if (C == 1) {
    qr_panel_reg2_kernel<QR_NB_REG, QR_REG_NT, QR_REG_RPT, false><<<1, QR_REG_NT, 0, st>>>(V, ld, m, j0, nbw, Vc, tau,
                                                                                          Tp, rpc);
    return cudaGetLastError();
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(C); cfg.blockDim = dim3(QR_REG_NT); cfg.dynamicSmemBytes = 0; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, qr_panel_reg2_kernel<QR_NB_REG, QR_REG_NT, QR_REG_RPT, true>, V, ld, m, j0, nbw, Vc,
                            tau, Tp, rpc);
}

// Y <- (I - Vp op(T) Vp^T) Y with the three WY kernels.  Returns launches.
template <int NB>
int apply_block_reflector(cudaStream_t st, const double* Vp, long long ldv, double* Y, long long ldy, long long rows,
                          int nc, int nbw, const double* Tp, int transT, const QrWork& wk) {
  int chunk = 32;
  long long nparts = (rows + chunk - 1) / chunk;
  if (nparts > QR_MAX_PARTS) { chunk = (int)((rows + QR_MAX_PARTS - 1) / QR_MAX_PARTS); nparts = (rows + chunk - 1) / chunk; }
  wy_partial_kernel<NB><<<(unsigned)nparts, 256, 0, st>>>(Vp, ldv, Y, ldy, rows, nc, nbw, chunk, wk.part);
  wy_reduce_kernel<NB><<<(nc + 3) / 4, 1024, 0, st>>>(wk.part, (int)nparts, nc, nbw, Tp, transT, wk.W2);
  wy_update_kernel<NB><<<(unsigned)nparts, 256, 0, st>>>(Vp, ldv, Y, ldy, rows, nc, nbw, chunk, wk.W2);
  return 3;
}

template <int NB>
long long form_q_global(cudaStream_t st, long long rows, int n, const QrWork& wk, double* Q, cudaError_t* err);

// Blocked Householder QR with compact-WY updates (K2a panel / K2b trailing / K2c form Q + sign fix).
template <int NB, bool REG>
long long qr_factor_blocked_t(cudaStream_t st, long long rows, int n, const double* X, double* Q, double* R,
                              void* work, cudaError_t* err) {
  QrWork wk;
  qr_layout(rows, n, static_cast<char*>(work), &wk);
  long long launches = 0;
  *err = cudaMemcpyAsync(wk.V, X, sizeof(double) * rows * n, cudaMemcpyDeviceToDevice, st);
  if (*err != cudaSuccess) return -1;
  // the clean reflectors are zero above their diagonal: rows above a panel are never written by its kernel
  *err = cudaMemsetAsync(wk.Vc, 0, sizeof(double) * rows * n, st);
  if (*err != cudaSuccess) return -1;
  const int npan = (n + NB - 1) / NB;
  for (int p = 0; p < npan; ++p) {
    const int j0 = p * NB, nbw = (n - j0 < NB) ? n - j0 : NB, n2 = n - j0 - nbw;
    double* Tp = wk.Tfac + (size_t)p * NB * NB;
    *err = REG ? launch_panel_reg(st, wk.V, n, rows, j0, nbw, wk.Vc, wk.tau, Tp)
               : launch_panel(st, wk.V, n, rows, j0, nbw, wk.Vc, wk.tau, Tp);
    if (*err != cudaSuccess) return -1;
    ++launches;
    if (n2 > 0)      // trailing update: A2 <- (I - Vp T^T Vp^T) A2
      launches += apply_block_reflector<NB>(st, wk.Vc + (long long)j0 * n + j0, n, wk.V + (long long)j0 * n + j0 + nbw,
                                            n, rows - j0, n2, nbw, Tp, 1, wk);
  }
  copy_triu_kernel<<<(n * n + 255) / 256, 256, 0, st>>>(wk.V, n, n, R);
  launches += 1;
  {
    // G = V^T V on the DMMA GEMM (split-K), then the one-shot form-Q
    int nl = launch_gemm(st, 0, GemmCall{wk.Vc, n, 1, wk.Vc, n, wk.Gq, plain_map(n), IndexMap{1, 1, 0}, n, n, (int)rows, 0},
                         wk.splitk, wk.splitk_elems, err);
    if (nl < 0) return -1;
    launches += nl;
    long long nq = form_q_global<NB>(st, rows, n, wk, Q, err);
    if (nq < 0) return -1;
    launches += nq;
  }
  sign_fix_kernel<<<296, 256, 0, st>>>(Q, rows, n, R);
  sign_fix_R_kernel<<<n, 128, 0, st>>>(R, n);
  launches += 2;
  *err = cudaGetLastError();
  return *err == cudaSuccess ? launches : -1;
}

// Form Q from the clean reflectors Vc, the Gram matrix G = V^T V (strict upper part) and the per-block T_p:
// Q = [I;0] - V X, (D^-1 + striu(G)) X = V_top^T  (see wy_formq_trsm_kernel).  Returns launches or -1.
template <int NB>
long long form_q_global(cudaStream_t st, long long rows, int n, const QrWork& wk, double* Q, cudaError_t* err) {
  long long launches = 0;
  const int npan = (n + NB - 1) / NB;
  static bool trsm_attr = false;
  if (!trsm_attr) {
    *err = cudaFuncSetAttribute(wy_formq_trsm_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (*err != cudaSuccess) return -1;
    trsm_attr = true;
  }
  set_identity_top_kernel<<<296, 256, 0, st>>>(Q, rows, n);
  wy_formq_trsm_kernel<NB><<<npan, NB * NB, sizeof(double) * (size_t)npan * NB * NB * 2, st>>>(wk.Gq, wk.Tfac, wk.Vc, n, n,
                                                                                             wk.Xq);
  transpose_tall_kernel<<<dim3((unsigned)((rows + 31) / 32), (n + 31) / 32), dim3(32, 8), 0, st>>>(wk.Vc, rows, n, wk.Vct);
  launches += 3;
  int nl = launch_gemm(st, 0, GemmCall{wk.Vct, rows, 1, wk.Xq, n, Q, plain_map(n), IndexMap{1, 1, 0}, (int)rows, n, n, 1},
                       wk.splitk, wk.splitk_elems, err);                                            // Q -= V X
  if (nl < 0) return -1;
  return launches + nl;
}

// Whole-matrix register-resident QR for small / medium c~ (n <= 112 columns, one cluster).  Returns -2 if it does not fit.
template <int NCS, int RPT>
long long qr_factor_fullreg_t(cudaStream_t st, long long rows, int n, const double* X, double* Q, double* R, const QrWork& wk,
                              cudaError_t* err) {
  constexpr int NP = NCS * 16, cap = RPT * 16;
  static int maxc = -1;
  constexpr size_t smem = sizeof(double) * (2 * 16 * NP + 2 * NP + 2 * 8 * NP + NP + NP * NP + 2 * NP);
  if (maxc < 0) {
    *err = cudaFuncSetAttribute(qr_full_reg_kernel<NCS, RPT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (*err != cudaSuccess) return -1;
    *err = cudaFuncSetAttribute(qr_full_reg_kernel<NCS, RPT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (*err != cudaSuccess) return -1;
    maxc = cudaFuncSetAttribute(qr_full_reg_kernel<NCS, RPT, true>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) ==
                   cudaSuccess ? 16 : 8;
    cudaGetLastError();
  }
  int C = 1;
  while (C < maxc && (rows + C - 1) / C > cap) C *= 2;
  const long long rpc = (rows + C - 1) / C;
  if (rpc > cap || (C > 1 && rpc < n)) return -2;           // too tall, or the diagonal rows would leave rank 0
  if (C == 1) {
    qr_full_reg_kernel<NCS, RPT, false><<<1, 256, smem, st>>>(X, (long long)n, rows, n, R, wk.Vc, wk.tau, wk.Gq, wk.Tfac, rpc);
  } else {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(C); cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    *err = cudaLaunchKernelEx(&cfg, qr_full_reg_kernel<NCS, RPT, true>, X, (long long)n, rows, n, R, wk.Vc, wk.tau, wk.Gq,
                              wk.Tfac, rpc);
    if (*err != cudaSuccess) return -1;
  }
  long long launches = 1;
  long long nq = form_q_global<16>(st, rows, n, wk, Q, err);
  if (nq < 0) return -1;
  launches += nq;
  sign_fix_kernel<<<296, 256, 0, st>>>(Q, rows, n, R);
  sign_fix_R_kernel<<<n, 128, 0, st>>>(R, n);
  launches += 2;
  *err = cudaGetLastError();
  return *err == cudaSuccess ? launches : -1;
}

// qr_path: 0 = automatic (whole-matrix register kernel when it fits, else blocked), 2 = always blocked
long long qr_factor_blocked(cudaStream_t st, int qr_path, long long rows, int n, const double* X, double* Q,
                            double* R, void* work, cudaError_t* err) {
  if (qr_path == 0 && n <= 112) {
    QrWork wk;
    qr_layout(rows, n, static_cast<char*>(work), &wk);
    long long nl = n <= 32 ? qr_factor_fullreg_t<2, 24>(st, rows, n, X, Q, R, wk, err)
                 : n <= 64 ? qr_factor_fullreg_t<4, 16>(st, rows, n, X, Q, R, wk, err)
                           : qr_factor_fullreg_t<7, 10>(st, rows, n, X, Q, R, wk, err);
    if (nl != -2) return nl;
  }
  constexpr long long cap = (long long)QR_REG_RPT * (QR_REG_NT / QR_NB_REG);
  if (rows <= cap * reg_panel_max_cluster())
    return qr_factor_blocked_t<QR_NB_REG, true>(st, rows, n, X, Q, R, work, err);
  return qr_factor_blocked_t<QR_NB, false>(st, rows, n, X, Q, R, work, err);
}

// ------------------------------------------------------------------ NEXT-2: top-k symmetric eigensolver
constexpr int EIGH_MAX_N = 14000;
constexpr int EIGH_MAX_GROUPS = 96;   // row groups of the tridiagonalisation sweep (column partials of y per group)     // d, e2 of the multisection / two columns of the back-transform in shared memory

struct EighWork {
  double *v0, *v1, *w, *y, *tau, *d, *e, *eig, *scal, *Z, *U0, *U1, *U2, *R, *rowpart, *colpart;
  void* qr;
};

size_t eigh_layout(long long n, int k, char* base, EighWork* w) {
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
  const size_t dbl = sizeof(double);
  size_t o[14];
  for (int i = 0; i < 8; ++i) o[i] = take(dbl * n);         // v0 v1 w y tau d e eig
  o[8] = take(dbl * 16);
  for (int i = 9; i < 13; ++i) o[i] = take(dbl * n * k);    // Z U0 U1 U2
  o[13] = take(dbl * (size_t)k * k);
  size_t oy = take(dbl * n * ((EIGH_MAX_N + EIGH_CW - 1) / EIGH_CW));
  size_t oc = take(dbl * n * EIGH_MAX_GROUPS);
  size_t oq = take(qr_work_bytes_impl(n, k));
  if (w) {
    w->rowpart = reinterpret_cast<double*>(base + oy);
    w->colpart = reinterpret_cast<double*>(base + oc);
    double** f[14] = {&w->v0, &w->v1, &w->w, &w->y, &w->tau, &w->d, &w->e, &w->eig, &w->scal,
                      &w->Z, &w->U0, &w->U1, &w->U2, &w->R};
    for (int i = 0; i < 14; ++i) *f[i] = reinterpret_cast<double*>(base + o[i]);
    w->qr = base + oq;
  }
  return off;
}

unsigned long long eigh_work_bytes_impl(long long n, int k) {
  if (n < 1 || k < 1 || k > n || n > EIGH_MAX_N) return 0;
  return eigh_layout(n, k, nullptr, nullptr);
}

// W (n x n symmetric, row-major, DEVICE, destroyed) -> lam[k] (largest |lambda| first), U (n x k, ld k).
// Returns kernels launched or -1.
long long eigh_top(cudaStream_t st, int n, int k, double* W, double* lam, double* U, void* work, cudaError_t* err) {
  EighWork wk;
  eigh_layout(n, k, static_cast<char*>(work), &wk);
  long long launches = 0;
  static int attr_done = 0;
  if (!attr_done) {
    int dev = 0, max_smem = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaFuncSetAttribute(multisect_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem - 1024);
    cudaFuncSetAttribute(eigh_backtransform_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem - 1024);
    attr_done = 1;
  }
  cudaMemsetAsync(wk.tau, 0, sizeof(double) * n, st);
#define REFL(k_, vprev_, vnew_)                                                                                  \
  do {                                                                                                           \
    const int left_ = n - (k_);                                                                                  \
    if (left_ <= 2048) eigh_reflector_kernel<2><<<1, 1024, 0, st>>>(W, n, (k_), wk.y, wk.rowpart, wk.colpart, rg_prev, (vprev_), wk.w, (vnew_), wk.tau, wk.d, wk.e); \
    else if (left_ <= 6144) eigh_reflector_kernel<6><<<1, 1024, 0, st>>>(W, n, (k_), wk.y, wk.rowpart, wk.colpart, rg_prev, (vprev_), wk.w, (vnew_), wk.tau, wk.d, wk.e); \
    else if (left_ <= 10240) eigh_reflector_kernel<10><<<1, 1024, 0, st>>>(W, n, (k_), wk.y, wk.rowpart, wk.colpart, rg_prev, (vprev_), wk.w, (vnew_), wk.tau, wk.d, wk.e); \
    else eigh_reflector_kernel<14><<<1, 1024, 0, st>>>(W, n, (k_), wk.y, wk.rowpart, wk.colpart, rg_prev, (vprev_), wk.w, (vnew_), wk.tau, wk.d, wk.e); \
  } while (0)
  int rg_prev = 0;                                 // > 0: the next reflector kernel sums the partials itself
  for (int k2 = 0; k2 + 2 < n; ++k2) {
    double* vprev = (k2 & 1) ? wk.v0 : wk.v1;      // v_{k-1}
    double* vnew = (k2 & 1) ? wk.v1 : wk.v0;       // v_k
    REFL(k2, vprev, vnew);
    const int nt = n - k2 - 1;                     // trailing block is nt x nt
    const int nch = (nt + EIGH_CW - 1) / EIGH_CW;
    // rows per group: a multiple of 32, about 600 CTAs in the upper triangle, at most EIGH_MAX_GROUPS groups
    long long G = (long long)nt * nch / (2 * 32 * 600);
    const long long gmin = (nt + 32LL * EIGH_MAX_GROUPS - 1) / (32LL * EIGH_MAX_GROUPS);
    if (G < gmin) G = gmin;
    if (G < 1) G = 1;
    const int rg = (int)(32 * G), ng = (nt + rg - 1) / rg;
    eigh_pass_kernel<<<dim3(nch, ng), 256, 0, st>>>(W, n, k2, rg, vprev, wk.w, vnew, wk.rowpart, wk.colpart);
    if (nt <= 2048) { rg_prev = rg; launches += 2; }       // launch-latency-bound tail: one kernel fewer per step
    else {
      eigh_ysum_kernel<<<(nt + 63) / 64, 64, 0, st>>>(wk.rowpart, wk.colpart, n, k2, rg, wk.y);
      rg_prev = 0; launches += 3;
    }
  }
  {
    const int kf = n >= 2 ? n - 2 : 0;
    double* vprev = (kf & 1) ? wk.v0 : wk.v1;
    REFL(kf, vprev, wk.v0);
    launches += 1;
  }
#undef REFL
  const int nc = 2 * k < n ? 2 * k : n;            // candidates: the k smallest and the k largest eigenvalues
  multisect_kernel<<<(nc + 7) / 8, 256, sizeof(double) * (2 * (size_t)n + 40), st>>>(wk.d, wk.e, n, wk.eig, k);
  eigh_select_kernel<<<(nc + 255) / 256, 256, 0, st>>>(wk.eig, nc, k, lam, wk.d, wk.e, n, wk.scal);
  eigh_invit_kernel<<<(k + 31) / 32, 32, 0, st>>>(wk.d, wk.e, n, lam, k, wk.scal, wk.Z, wk.U0, wk.U1, wk.U2, 3);
  launches += 4;
  *err = cudaGetLastError();
  if (*err != cudaSuccess) return -1;
  long long nq = qr_factor_blocked(st, 0, n, k, wk.Z, U, wk.R, wk.qr, err);
  if (nq < 0) return -1;
  launches += nq;
  if (n >= 3) {
    const int nb = (k + 1) / 2;
    eigh_backtransform_kernel<<<nb, 1024, sizeof(double) * 2 * (size_t)n, st>>>(W, wk.tau, n, U, k, k);
    launches += 1;
  }
  eigh_sign_kernel<<<k, 256, 0, st>>>(U, n, k);
  launches += 1;
  *err = cudaGetLastError();
  return *err == cudaSuccess ? launches : -1;
}

}  // namespace

// ------------------------------------------------------------------ step stages
namespace {

#define GEMM(h, call_)                                                                          \
  do {                                                                                          \
    cudaError_t ge__;                                                                           \
    int nl__ = launch_gemm((h)->stream, (h)->gemm_path, (call_), (h)->splitk, (h)->L.splitk_elems, &ge__); \
    if (nl__ < 0) return fail((h), QRCTM_ERR_CUDA, "gemm launch", ge__);                        \
    (h)->launches += nl__;                                                                      \
  } while (0)

// K1 (E1): X[(j,u),k] = sum_i C[j,i] T[i,u,k]       -> out (chi x b*chi == chi*b x chi)
// Computed transposed, X^T[(u,k), j] = sum_i T[i,(u,k)] C[i,j]^T, so that both operands are K x (M|N)
// row-major (bulk-copy kernel) and the long index is the GEMM's M; the epilogue writes X itself.
// Ct is C^T as a K x N matrix: C itself when it is exactly symmetric (SYMMETRIZE = 1).
int stage_reduced_corner(qrctm* h, const double* C, const double* T, double* X) {
  const int chi = h->chi; const long long bc = (long long)h->b * chi;
  if (h->symmetrize) {
    GemmCall c{T, bc, 1, C, chi, X, IndexMap{1, 1, 0}, plain_map(bc), (int)bc, chi, chi, 0};
    GEMM(h, c);
  } else {
    GemmCall c{C, chi, 0, T, bc, X, plain_map(bc), IndexMap{1, 1, 0}, chi, (int)bc, chi, 0};
    GEMM(h, c);
  }
  return QRCTM_OK;
}

// K3: P'[u,l,J,m] = sum_j Qm[j,u,m] T[j,l,J]        (Qm: chi*b x n viewed chi x b*n).  m innermost: the
// consecutive rows of a K4 tile (M index (J,m)) are then adjacent in K4's outputs.
// co = number of columns of Qm (the new chi) when it differs from the chi of T (eigen step with chi growth).
int stage_half_absorb(qrctm* h, const double* Qm, const double* T, double* P, int co = 0) {
  const int ci = h->chi, b = h->b; if (co <= 0) co = ci;
  const long long cc = (long long)ci * co;
  GemmCall c{Qm, (long long)b * co, 1, T, (long long)b * ci, P, IndexMap{co, b * cc, 1}, IndexMap{ci, cc, co},
             b * co, b * ci, ci, 0};
  GEMM(h, c);
  return QRCTM_OK;
}

// K4: S[m,J,d,r] = sum_{u,l} P'[(u,l),(J,m)] a[(u,l),(d,r)]      (GEMM row index i = J*chi + m)
//   layout 0: S''[J,d,m,r]  (what K5 wants: K x M with K = (J,d))
//   layout 1: S~ [m,r,J,d]  (what the kappa network wants: K = (m,r))
//   layout 2: C~[(J,d),(m,r)] natural enlarged-corner matrix == layout 0
int stage_absorb_a(qrctm* h, const double* P, double* S, int layout, const double* amat = nullptr, int chi_out = 0) {
  const int ci = h->chi, chi = chi_out > 0 ? chi_out : ci, b = h->b;     // chi: range of the index m
  const long long m = (long long)chi * b, cc = (long long)ci * chi;
  IndexMap ro, co;
  if (layout == 0) { ro = IndexMap{chi, (long long)b * m, b}; co = IndexMap{b, m, 1}; }
  else             { ro = IndexMap{chi, b, (long long)b * m}; co = IndexMap{b, 1, (long long)chi * b}; }
  GemmCall c{P, cc, 1, amat ? amat : h->a_mat, h->L.lda_a, S, ro, co, (int)cc, b * b, b * b, 0};
  c.epi = 1;
  GEMM(h, c);
  return QRCTM_OK;
}

// K4 layered (NEXT-1): the same S'' without ever using the double-layer tensor,
//   P1[(s,u_b,l_b)][J,d_k,m,r_k] = sum_{u_k,l_k} P'[(u_k u_b),(l_k l_b),J,m] A[s,u_k,l_k,d_k,r_k]   (D^2 batched GEMMs, K = D^2)
//   S''[J,(d_k d_b),m,(r_k r_b)] = sum_{s,u_b,l_b} P1[(s,u_b,l_b)][J,d_k,m,r_k] A[s,u_b,l_b,d_b,r_b]  (K = d D^2)
// 4 d chi^2 D^6 flops instead of 2 chi^2 D^8.  Needs even chi (16-byte aligned rows for the bulk copies).
bool layered_ok(const qrctm* h) { return h->chi % 2 == 0; }

int stage_absorb_layered(qrctm* h, const double* P, double* S) {
  const int chi = h->chi, D = h->D, b = h->b, d = h->d;
  const long long m = h->m, cc = (long long)chi * chi, M2 = cc * b;
  GemmCall g1{P, cc, 1, h->B1, h->L.ld1, h->P1,
              IndexMap{chi, (long long)D * chi * D, D},
              IndexMap{D * D, (long long)b * M2, (long long)chi * D, D, 1},
              (int)cc, d * b, b, 0};
  g1.ka = IndexMap{D, (long long)D * b, D};
  g1.batch = b;
  g1.za = IndexMap{D, (long long)b * cc, cc};
  g1.zo = M2;
  g1.epi = 1;
  GEMM(h, g1);
  GemmCall g2{h->P1, M2, 1, h->B2, h->L.ld2, S, IndexMap{chi * D, (long long)D * m, D}, IndexMap{D, m, 1},
              (int)M2, b, d * b, 0};
  g2.epi = 1;
  GEMM(h, g2);
  return QRCTM_OK;
}

// K5: out[(m,r),n] = sum_{(J,d)} S''[(J,d),(m,r)] Qm[(J,d),n]
// chi_out: range of the index m of S'' (rows of out / D^2); ncols: columns of Qm (default: chi_out).
int stage_project(qrctm* h, const double* S, const double* Qm, double* out, int chi_out = 0, int ncols = 0) {
  const int chi = chi_out > 0 ? chi_out : h->chi; const long long m = (long long)chi * h->b, mi = h->m;
  const int nq = ncols > 0 ? ncols : chi;
  GemmCall c{S, m, 1, Qm, nq, out, plain_map(nq), IndexMap{1, 1, 0}, (int)m, nq, (int)mi, 0};
  c.epi = 1;
  GEMM(h, c);
  return QRCTM_OK;
}

// K6 (E4): W[m,(r,n)] = sum_k R[m,k] Q[k,(r,n)] ;  C'[p,n] = sum_{(m,r)} T'[(m,r),p] W[(m,r),n]
int stage_corner_accel(qrctm* h) {
  const int chi = h->chi; const long long bc = (long long)h->b * chi, m = h->m;
  // W^T[(r,n), m] = sum_k Q[k,(r,n)] R^T[k,m]  (long index as M, both operands K-major); writes W
  transpose_small_kernel<<<(chi * chi + 255) / 256, 256, 0, h->stream>>>(h->R, chi, h->Rt);
  h->launches += 1;
  GemmCall c1{h->Q, bc, 1, h->Rt, chi, h->W, IndexMap{1, 1, 0}, plain_map(bc), (int)bc, chi, chi, 0};
  GEMM(h, c1);
  GemmCall c2{h->Tn, chi, 1, h->W, chi, h->Cn, plain_map(chi), IndexMap{1, 1, 0}, chi, chi, (int)m, 0};
  GEMM(h, c2);
  return QRCTM_OK;
}

// K6' (E5)+(E4'): Z = half_absorb(X), C~ = Z.a, Y = C~ Q, C' = Q^T Y
int stage_corner_enlarged(qrctm* h) {
  const int chi = h->chi; const long long m = h->m;
  int rc = stage_half_absorb(h, h->X, h->T, h->P); if (rc) return rc;
  rc = stage_absorb_a(h, h->P, h->S, 0); if (rc) return rc;          // S = C~[(J,d),(k,r)]
  GemmCall c1{h->S, m, 0, h->Q, chi, h->W, plain_map(chi), IndexMap{1, 1, 0}, (int)m, chi, (int)m, 0};
  GEMM(h, c1);
  GemmCall c2{h->Q, chi, 1, h->W, chi, h->Cn, plain_map(chi), IndexMap{1, 1, 0}, chi, chi, (int)m, 0};
  GEMM(h, c2);
  return QRCTM_OK;
}

// K7: C,T <- sym(Cn,Tn) / ||.||_F
int stage_normalize(qrctm* h, const double* Cn, const double* Tn) {
  const int chi = h->chi, b = h->b;
  long long nT = (long long)chi * b * chi;
  int nbC = (int)(((long long)chi * chi + 255) / 256); if (nbC > 148) nbC = 148;
  int nbT = (int)((nT + 255) / 256); if (nbT > kPartialBlocks) nbT = kPartialBlocks;
  sym_partial_kernel<<<nbC + nbT, 256, 0, h->stream>>>(Cn, Tn, chi, b, h->symmetrize, h->C, h->T, h->partial,
                                                      nbC, nbT);
  int nb = (int)((nT + (long long)chi * chi + 255) / 256); if (nb > 592) nb = 592;
  scale_kernel<<<nb, 256, 0, h->stream>>>(h->C, h->T, chi, b, h->partial, nbC, nbT, h->scal, h->flag);
  h->launches += 2;
  CU(h, cudaGetLastError());
  return QRCTM_OK;
}

// K8: spectrum of h->C into s_out (+ delta against s_prev, optional update)
int stage_spectrum(qrctm* h, double* s_out, int update_prev, cudaStream_t st) {
  const int chi = h->chi;
  static int max_smem = -1;
  if (max_smem < 0) {
    int dev = 0; cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    max_smem -= 1024;      // static shared memory of the kernel
    CU(h, cudaFuncSetAttribute(tridiag_smem_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));
  }
  const size_t tri_bytes = sizeof(double) * ((size_t)chi * (chi + 1) / 2 + 2 * (size_t)chi + 40);
  const int nt = ((chi + 31) / 32 * 32) < 64 ? 64 : (chi + 31) / 32 * 32;
  if (tri_bytes <= (size_t)max_smem && chi <= 1024) {
    tridiag_smem_kernel<<<1, 1024, tri_bytes, st>>>(h->C, chi, h->dvec, h->evec);
    multisect_kernel<<<(chi + 7) / 8, 256, sizeof(double) * (2 * chi + 40), st>>>(h->dvec, h->evec, chi,
                                                                                         h->eig);
    spectrum_finalize_kernel<<<1, nt, sizeof(double) * (chi + 40), st>>>(h->eig, chi, s_out, h->s_prev,
                                                                                 h->delta, update_prev);
    h->launches += 3;
  } else {
    CU(h, cudaMemcpyAsync(h->Wc, h->C, sizeof(double) * chi * chi, cudaMemcpyDeviceToDevice, st));
    tridiag_kernel<<<1, 1024, 0, st>>>(h->Wc, chi, h->dvec, h->evec, h->vv, h->pv);
    bisect_sort_kernel<<<1, nt, sizeof(double) * (3 * chi + 40), st>>>(h->dvec, h->evec, chi, h->eig, s_out,
                                                                            h->s_prev, h->delta, update_prev);
    h->launches += 2;
  }
  CU(h, cudaGetLastError());
  return QRCTM_OK;
}

int do_step(qrctm* h, cudaEvent_t* ev /* QRCTM_NSTAGE+1 events or null */, bool with_k7 = true) {
  // NVTX ranges name the stages so that `ncu --nvtx --nvtx-include "K4_absorb_a/"` selects one.
  auto mark = [&](int i, const char* next) {
    if (i > 0) nvtxRangePop();
    if (ev) cudaEventRecord(ev[i], h->stream);
    if (next) nvtxRangePushA(next);
  };
  int rc = QRCTM_OK;
  mark(0, "K1_reduced_corner");
  rc = stage_reduced_corner(h, h->C, h->T, h->X);
  if (!rc) {
    mark(1, "K2_qr");
    cudaError_t e;
    long long nl = h->qr_path != 1
        ? qr_factor_blocked(h->stream, h->qr_path, h->m, h->chi, h->X, h->Q, h->R, h->qrwork, &e)
        : qr_factor_level2(h->stream, h->m, h->chi, h->X, h->Q, h->R, h->qrwork, &e);
    if (nl < 0) rc = fail(h, QRCTM_ERR_CUDA, "qr", e); else h->launches += nl;
  }
  if (!rc) { mark(2, "K3_half_absorb"); rc = stage_half_absorb(h, h->Q, h->T, h->P); }
  if (!rc) {
    mark(3, "K4_absorb_a");
    rc = (h->absorb_mode == 1 && layered_ok(h)) ? stage_absorb_layered(h, h->P, h->S) : stage_absorb_a(h, h->P, h->S, 0);
  }
  if (!rc) { mark(4, "K5_project"); rc = stage_project(h, h->S, h->Q, h->Tn); }
  if (!rc) { mark(5, "K6_corner"); rc = h->corner_mode == 0 ? stage_corner_accel(h) : stage_corner_enlarged(h); }
  if (!rc && !with_k7) { nvtxRangePop(); return rc; }
  if (!rc) { mark(6, "K7_normalize"); rc = stage_normalize(h, h->Cn, h->Tn); }
  if (!rc) mark(7, nullptr); else nvtxRangePop();
  return rc;
}

void invalidate_graphs(qrctm* h) {
  if (h->g_front) { cudaGraphExecDestroy(h->g_front); h->g_front = nullptr; }
  if (h->g_k7) { cudaGraphExecDestroy(h->g_k7); h->g_k7 = nullptr; }
  h->graph_failed = 0;
  h->warm_steps = 0;      // one ordinary step first: newly selected kernels set their attributes outside capture
}

// current bond dimension (NEXT-2 warm-up grows it up to chi_cap); captured graphs hold the old shapes
void set_chi(qrctm* h, int chi) {
  if (chi == h->chi) return;
  invalidate_graphs(h);
  h->chi = chi; h->m = (long long)chi * h->b;
}

// Capture `body` (which only enqueues work on h->stream) into an executable graph.
template <class F>
bool capture_graph(qrctm* h, F body, cudaGraphExec_t* exec, long long* nlaunch) {
  const long long l0 = h->launches;
  if (cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) { cudaGetLastError(); return false; }
  const int rc = body();
  cudaGraph_t graph = nullptr;
  cudaError_t e = cudaStreamEndCapture(h->stream, &graph);
  *nlaunch = h->launches - l0;
  h->launches = l0;
  if (rc != QRCTM_OK || e != cudaSuccess || !graph) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return false; }
  e = cudaGraphInstantiate(exec, graph, 0);
  cudaGraphDestroy(graph);
  if (e != cudaSuccess) { *exec = nullptr; cudaGetLastError(); return false; }
  return true;
}

// K1..K6 (front) and K7, replayed from CUDA graphs once one ordinary step has run (so that all
// one-time function attributes are set) -- unless events / NVTX ranges per stage are wanted.
int run_front(qrctm* h, cudaEvent_t* ev) {
  const bool can = h->use_graph && !ev && h->stream != nullptr && !h->graph_failed && h->warm_steps >= 1;
  if (can && !h->g_front) {
    if (!capture_graph(h, [&] { return do_step(h, nullptr, false); }, &h->g_front, &h->g_front_n)) h->graph_failed = 1;
  }
  if (can && h->g_front) {
    CU(h, cudaGraphLaunch(h->g_front, h->stream));
    h->launches += h->g_front_n;
    return QRCTM_OK;
  }
  return do_step(h, ev, false);
}

int run_k7(qrctm* h, cudaEvent_t* ev) {
  const bool can = h->use_graph && !ev && h->stream != nullptr && !h->graph_failed && h->warm_steps >= 1;
  if (can && !h->g_k7) {
    if (!capture_graph(h, [&] { return stage_normalize(h, h->Cn, h->Tn); }, &h->g_k7, &h->g_k7_n)) h->graph_failed = 1;
  }
  int rc;
  if (can && h->g_k7) {
    CU(h, cudaGraphLaunch(h->g_k7, h->stream));
    h->launches += h->g_k7_n;
    rc = QRCTM_OK;
  } else {
    if (ev) { nvtxRangePushA("K7_normalize"); cudaEventRecord(ev[6], h->stream); }
    rc = stage_normalize(h, h->Cn, h->Tn);
    if (ev) { cudaEventRecord(ev[7], h->stream); nvtxRangePop(); }
  }
  if (rc == QRCTM_OK) h->warm_steps += 1;
  return rc;
}

int check_flag(qrctm* h) {   // stream must be synchronised by the caller's copy
  CU(h, cudaMemcpyAsync(h->h_flag, h->flag, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  if (*h->h_flag) return fail(h, QRCTM_ERR_NUMERIC, "NaN/Inf or zero Frobenius norm in C' or T'");
  return QRCTM_OK;
}

}  // namespace

// ------------------------------------------------------------------ C ABI
extern "C" {

const char* qrctm_version(void) { return "qrctm-b200 0.1 (sm_100a, FP64 DMMA)"; }

unsigned long long qrctm_workspace_bytes(int d, int D, int chi) {
  Layout L;
  if (!make_layout(d, D, chi, &L)) return 0;
  return L.total;
}

static int create_common(int d, int D, int chi, void* ws, unsigned long long ws_bytes, qrctm_t** out) {
  if (!out) return QRCTM_ERR_INVALID_ARG;
  *out = nullptr;
  Layout L;
  if (!make_layout(d, D, chi, &L)) return QRCTM_ERR_INVALID_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return QRCTM_ERR_CUDA; }
  qrctm* h = new (std::nothrow) qrctm();
  if (!h) return QRCTM_ERR_CUDA;
  memset(h, 0, sizeof(*h));
  h->d = d; h->D = D; h->b = D * D; h->chi = chi; h->m = (long long)chi * D * D;
  h->chi_cap = chi; h->eigwork = nullptr; h->eigwork_bytes = 0; h->eig_rows = h->eig_cols = 0;
  h->L = L; h->stream = 0;
  h->corner_mode = 0; h->symmetrize = 1; h->check_every = 1; h->gemm_path = 0; h->overlap = 1; h->use_graph = 1;
  if (ws) {
    if (ws_bytes < L.total || (reinterpret_cast<uintptr_t>(ws) & (kAlign - 1)) || !is_device_ptr(ws)) {
      delete h; return QRCTM_ERR_INVALID_ARG;
    }
    h->base = static_cast<char*>(ws); h->owns_ws = false;
  } else {
    void* p = nullptr;
    if (cudaMalloc(&p, L.total) != cudaSuccess) { cudaGetLastError(); delete h; return QRCTM_ERR_CUDA; }
    h->base = static_cast<char*>(p); h->owns_ws = true;
  }
  bind_views(h);
  void* hp = nullptr;
  if (cudaMallocHost(&hp, 64 * sizeof(double)) != cudaSuccess) {
    cudaGetLastError(); if (h->owns_ws) cudaFree(h->base); delete h; return QRCTM_ERR_CUDA;
  }
  h->h_pinned = static_cast<double*>(hp);
  {
    int lo = 0, hi = 0;
    cudaDeviceGetStreamPriorityRange(&lo, &hi);
    if (cudaStreamCreateWithPriority(&h->side, cudaStreamNonBlocking, hi) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_env, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_spec, cudaEventDisableTiming) != cudaSuccess) {
      cudaGetLastError(); h->side = nullptr; h->overlap = 0;
    }
  }
  h->h_flag = reinterpret_cast<int*>(h->h_pinned + 32);       // [64..319] holds the two-site RDM
  cudaMemsetAsync(h->flag, 0, 4 * sizeof(int), 0);
  {   // padded operand matrices: the pad columns are zeroed once and never written again
    const size_t b2 = (size_t)h->b * h->b;
    cudaMemsetAsync(h->a_mat, 0, sizeof(double) * b2 * L.lda_a, 0);
    cudaMemsetAsync(h->a2_mat, 0, sizeof(double) * b2 * L.lda_a, 0);
    cudaMemsetAsync(h->B1, 0, sizeof(double) * h->b * L.ld1, 0);
    cudaMemsetAsync(h->B2, 0, sizeof(double) * (size_t)d * h->b * L.ld2, 0);
  }
  cudaMemsetAsync(h->s_prev, 0, sizeof(double) * chi, 0);
  cudaMemsetAsync(h->R, 0, sizeof(double) * chi * chi, 0);
  cudaMemsetAsync(h->Q, 0, sizeof(double) * h->m * chi, 0);
  if (cudaStreamSynchronize(0) != cudaSuccess) { cudaGetLastError(); qrctm_destroy(h); return QRCTM_ERR_CUDA; }
  *out = h;
  return QRCTM_OK;
}

int qrctm_create(int d, int D, int chi, qrctm_t** out) { return create_common(d, D, chi, nullptr, 0, out); }

int qrctm_create_in(int d, int D, int chi, void* workspace, unsigned long long workspace_bytes, qrctm_t** out) {
  if (!workspace) return QRCTM_ERR_INVALID_ARG;
  return create_common(d, D, chi, workspace, workspace_bytes, out);
}

int qrctm_destroy(qrctm_t* h) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  cudaStreamSynchronize(h->stream);
  invalidate_graphs(h);
  if (h->owns_ws && h->base) cudaFree(h->base);
  if (h->eigwork) cudaFree(h->eigwork);
  if (h->h_pinned) cudaFreeHost(h->h_pinned);
  if (h->side) { cudaStreamSynchronize(h->side); cudaStreamDestroy(h->side); cudaEventDestroy(h->ev_env); cudaEventDestroy(h->ev_spec); }
  if (h->have_ev) for (int i = 0; i < QRCTM_NSTAGE + 2; ++i) cudaEventDestroy(h->ev[i]);
  cudaGetLastError();
  delete h;
  return QRCTM_OK;
}

int qrctm_set_stream(qrctm_t* h, void* cuda_stream) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  CU(h, cudaStreamSynchronize(h->stream));
  invalidate_graphs(h);
  h->stream = static_cast<cudaStream_t>(cuda_stream);
  return QRCTM_OK;
}

int qrctm_set_A(qrctm_t* h, const double* A) {
  if (!h || !A) return h ? fail(h, QRCTM_ERR_INVALID_ARG, "null A") : QRCTM_ERR_INVALID_ARG;
  long long b2 = (long long)h->b * h->b;
  CU(h, copy_in(h->A, A, (size_t)h->d * b2, h->stream));
  build_a_kernel<<<(unsigned)b2, 256, 0, h->stream>>>(h->A, h->d, h->D, h->a_mat, h->L.lda_a);
  build_layers_kernel<<<64, 256, 0, h->stream>>>(h->A, h->d, h->D, h->B1, h->L.ld1, h->B2, h->L.ld2);
  h->launches += 2;
  CU(h, cudaGetLastError());
  h->have_A = true;
  return QRCTM_OK;
}

int qrctm_set_env(qrctm_t* h, const double* C, const double* T) {
  if (!h || !C || !T) return h ? fail(h, QRCTM_ERR_INVALID_ARG, "null C/T") : QRCTM_ERR_INVALID_ARG;
  if (h->chi != h->chi_cap) { CU(h, cudaStreamSynchronize(h->stream)); set_chi(h, h->chi_cap); }
  CU(h, copy_in(h->Cn, C, (size_t)h->chi * h->chi, h->stream));
  CU(h, copy_in(h->Tn, T, (size_t)h->m * h->chi, h->stream));
  CU(h, cudaMemsetAsync(h->flag, 0, sizeof(int), h->stream));
  int rc = stage_normalize(h, h->Cn, h->Tn); if (rc) return rc;
  rc = check_flag(h); if (rc) return rc;
  CU(h, cudaMemsetAsync(h->s_prev, 0, sizeof(double) * h->chi, h->stream));
  h->need_s0 = 1;      // s_prev = spectrum(C0) is computed by the next qrctm_run, overlapped with its first step
  h->have_env = true;
  return QRCTM_OK;
}

int qrctm_step(qrctm_t* h) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (!h->have_A || !h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "set_A and set_env first");
  h->eig_rows = 0;          // Q is about to be overwritten by K2
  if (!h->use_graph || h->stream == nullptr) { int rc0 = do_step(h, nullptr); if (!rc0) h->warm_steps += 1; return rc0; }
  int rc = run_front(h, nullptr); if (rc) return rc;
  return run_k7(h, nullptr);
}

int qrctm_run(qrctm_t* h, int max_iter, double tol, int* iters_done, double* final_delta) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (!h->have_A || !h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "set_A and set_env first");
  h->eig_rows = 0;          // Q is about to be overwritten by K2
  if (max_iter < 0) return fail(h, QRCTM_ERR_INVALID_ARG, "max_iter < 0");
  if (h->overlap && h->side && !h->time_stages) {
    // Overlapped driver: K1..K6 of step it are queued before the host waits for the spectrum of
    // step it-1 (side stream); K7 of step it (the only stage that overwrites C, T) waits for it.
    double delta = INFINITY;
    int done = 0;
    bool pending = false;                       // a spectrum result is in flight on the side stream
    bool s0_inflight = false;
    if (h->need_s0 && max_iter > 0) {           // s_prev = spectrum(C0) on the side stream, under step 1's K1..K6
      CU(h, cudaEventRecord(h->ev_env, h->stream));
      CU(h, cudaStreamWaitEvent(h->side, h->ev_env, 0));
      int rc0 = stage_spectrum(h, h->s, 1, h->side); if (rc0) return rc0;
      CU(h, cudaEventRecord(h->ev_spec, h->side));
      h->need_s0 = 0; s0_inflight = true;
    }
    for (int it = 1; it <= max_iter; ++it) {
      int rc = run_front(h, nullptr); if (rc) return rc;
      if (s0_inflight) { CU(h, cudaStreamWaitEvent(h->stream, h->ev_spec, 0)); s0_inflight = false; }   // K7 overwrites C
      if (pending) {
        CU(h, cudaEventSynchronize(h->ev_spec));
        pending = false;
        if (h->h_flag[0]) { cudaStreamSynchronize(h->stream); return fail(h, QRCTM_ERR_NUMERIC, "NaN/Inf or zero Frobenius norm in C' or T'"); }
        delta = h->h_pinned[0];
        if (delta < tol) break;                 // converged at step it-1: the half step in flight is discarded
      }
      rc = run_k7(h, nullptr); if (rc) return rc;
      done = it;
      if (it % h->check_every == 0 || it == max_iter) {
        CU(h, cudaEventRecord(h->ev_env, h->stream));
        CU(h, cudaStreamWaitEvent(h->side, h->ev_env, 0));
        rc = stage_spectrum(h, h->s, 1, h->side); if (rc) return rc;
        CU(h, cudaMemcpyAsync(h->h_pinned, h->delta, sizeof(double), cudaMemcpyDeviceToHost, h->side));
        CU(h, cudaMemcpyAsync(h->h_flag, h->flag, sizeof(int), cudaMemcpyDeviceToHost, h->side));
        CU(h, cudaEventRecord(h->ev_spec, h->side));
        // (the next K7, the only writer of C, is enqueued after the host has seen ev_spec complete)
        pending = true;
      }
    }
    if (pending) {
      CU(h, cudaEventSynchronize(h->ev_spec));
      if (h->h_flag[0]) { cudaStreamSynchronize(h->stream); return fail(h, QRCTM_ERR_NUMERIC, "NaN/Inf or zero Frobenius norm in C' or T'"); }
      delta = h->h_pinned[0];
    }
    CU(h, cudaStreamSynchronize(h->stream));
    if (iters_done) *iters_done = done;
    if (final_delta) *final_delta = delta;
    return QRCTM_OK;
  }
  if (h->need_s0 && max_iter > 0) { int rc0 = stage_spectrum(h, h->s, 1, h->stream); if (rc0) return rc0; h->need_s0 = 0; }
  double delta = INFINITY;
  int it = 0;
  if (h->time_stages && !h->have_ev) {
    for (int i = 0; i < QRCTM_NSTAGE + 2; ++i) CU(h, cudaEventCreate(&h->ev[i]));
    h->have_ev = true;
  }
  for (it = 1; it <= max_iter; ++it) {
    int rc = do_step(h, h->time_stages ? h->ev : nullptr); if (rc) return rc;
    h->warm_steps += 1;
    const bool check = (it % h->check_every == 0 || it == max_iter);
    if (check) {
      rc = stage_spectrum(h, h->s, 1, h->stream); if (rc) return rc;
      CU(h, cudaMemcpyAsync(h->h_pinned, h->delta, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    }
    if (h->time_stages) CU(h, cudaEventRecord(h->ev[QRCTM_NSTAGE + 1], h->stream));
    if (check) { rc = check_flag(h); if (rc) return rc; }       // synchronises
    else if (h->time_stages) CU(h, cudaStreamSynchronize(h->stream));
    if (h->time_stages) {
      for (int i = 0; i <= QRCTM_NSTAGE; ++i) {
        float ms = 0.f;
        CU(h, cudaEventElapsedTime(&ms, h->ev[i], h->ev[i + 1]));
        h->stage_ms[i] += ms;
      }
      h->stage_steps += 1;
    }
    if (check) {
      delta = h->h_pinned[0];
      if (delta < tol) break;
    }
  }
  if (it > max_iter) it = max_iter;
  CU(h, cudaStreamSynchronize(h->stream));
  if (iters_done) *iters_done = it;
  if (final_delta) *final_delta = delta;
  return QRCTM_OK;
}

int qrctm_get_env(qrctm_t* h, double* C, double* T) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (!h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "no environment");
  int rc = check_flag(h); if (rc) return rc;
  if (C) CU(h, copy_out(C, h->C, (size_t)h->chi * h->chi, h->stream));
  if (T) CU(h, copy_out(T, h->T, (size_t)h->m * h->chi, h->stream));
  return QRCTM_OK;
}

int qrctm_get_corner_spectrum(qrctm_t* h, double* s) {
  if (!h || !s) return h ? fail(h, QRCTM_ERR_INVALID_ARG, "null s") : QRCTM_ERR_INVALID_ARG;
  if (!h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "no environment");
  int rc = stage_spectrum(h, h->s_tmp, 0, h->stream); if (rc) return rc;
  CU(h, copy_out(s, h->s_tmp, h->chi, h->stream));
  return QRCTM_OK;
}

int qrctm_get_qr(qrctm_t* h, double* Q, double* R) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (Q) CU(h, copy_out(Q, h->Q, (size_t)h->m * h->chi, h->stream));
  if (R) CU(h, copy_out(R, h->R, (size_t)h->chi * h->chi, h->stream));
  return QRCTM_OK;
}

int qrctm_get_raw(qrctm_t* h, double* Cn, double* Tn) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (Cn) CU(h, copy_out(Cn, h->Cn, (size_t)h->chi * h->chi, h->stream));
  if (Tn) CU(h, copy_out(Tn, h->Tn, (size_t)h->m * h->chi, h->stream));
  return QRCTM_OK;
}

int qrctm_get_a(qrctm_t* h, double* a) {
  if (!h || !a) return QRCTM_ERR_INVALID_ARG;
  if (!h->have_A) return fail(h, QRCTM_ERR_NOT_READY, "no A");
  long long b2 = (long long)h->b * h->b;
  cudaMemcpyKind k = is_device_ptr(a) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  CU(h, cudaMemcpy2DAsync(a, sizeof(double) * b2, h->a_mat, sizeof(double) * h->L.lda_a, sizeof(double) * b2, b2,
                          k, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  return QRCTM_OK;
}

int qrctm_set_option(qrctm_t* h, int key, int value) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  cudaStreamSynchronize(h->stream);
  invalidate_graphs(h);
  switch (key) {
    case QRCTM_OPT_CORNER_MODE: if (value != 0 && value != 1) break; h->corner_mode = value; return QRCTM_OK;
    case QRCTM_OPT_SYMMETRIZE:  if (value != 0 && value != 1) break; h->symmetrize = value; return QRCTM_OK;
    case QRCTM_OPT_CHECK_EVERY: if (value < 1) break; h->check_every = value; return QRCTM_OK;
    case QRCTM_OPT_GEMM_PATH:   if (value != 0 && value != 1) break; h->gemm_path = value; return QRCTM_OK;
    case QRCTM_OPT_QR_PATH:     if (value < 0 || value > 2) break; h->qr_path = value; return QRCTM_OK;
    case QRCTM_OPT_OVERLAP_CHECK: if (value != 0 && value != 1) break; h->overlap = value; return QRCTM_OK;
    case QRCTM_OPT_ABSORB_MODE: if (value != 0 && value != 1) break; h->absorb_mode = value; return QRCTM_OK;
    case QRCTM_OPT_USE_GRAPH:   if (value != 0 && value != 1) break; h->use_graph = value; return QRCTM_OK;
    case QRCTM_OPT_TIME_STAGES: if (value != 0 && value != 1) break; h->time_stages = value; return QRCTM_OK;
    default: break;
  }
  return fail(h, QRCTM_ERR_INVALID_ARG, "bad option key/value");
}

long long qrctm_launch_count(const qrctm_t* h) { return h ? h->launches : 0; }

int qrctm_get_stage_ms(qrctm_t* h, double* ms, long long* steps, int reset) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (ms) for (int i = 0; i <= QRCTM_NSTAGE; ++i) ms[i] = h->stage_ms[i];
  if (steps) *steps = h->stage_steps;
  if (reset) { for (int i = 0; i <= QRCTM_NSTAGE; ++i) h->stage_ms[i] = 0.0; h->stage_steps = 0; }
  return QRCTM_OK;
}

const char* qrctm_last_error(const qrctm_t* h) { return h ? h->err : "null handle"; }

}  // extern "C"

// ------------------------------------------------------------------ observables, diagnostics, stand-alone entries
#include "probe.cuh"

namespace {

__global__ void r_diag_minmax_kernel(const double* __restrict__ R, int n, double* __restrict__ out) {
  __shared__ double sh[33];
  double mn = INFINITY, mx = -INFINITY;
  for (int k = threadIdx.x; k < n; k += blockDim.x) {
    double v = R[(long long)k * n + k];
    mn = fmin(mn, v); mx = fmax(mx, v);
  }
  double gmx = block_max(mx, sh);
  double gmn = -block_max(-mn, sh);
  if (threadIdx.x == 0) { out[0] = gmn; out[1] = gmx; }
}

int reduce_dot(qrctm* h, const double* x, const double* y, long long n, double* out) {
  dot_partial_kernel<<<kPartialBlocks, 256, 0, h->stream>>>(x, y, n, h->partial + 2 * kPartialBlocks);
  sum_partial_kernel<<<1, 256, 0, h->stream>>>(h->partial + 2 * kPartialBlocks, kPartialBlocks, out);
  h->launches += 2;
  CU(h, cudaGetLastError());
  return QRCTM_OK;
}

}  // namespace

extern "C" {

int qrctm_norm_per_site(qrctm_t* h, double* kappa) {
  if (!h || !kappa) return h ? fail(h, QRCTM_ERR_INVALID_ARG, "null kappa") : QRCTM_ERR_INVALID_ARG;
  if (!h->have_A || !h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "set_A and set_env first");
  const int chi = h->chi; const long long m = h->m;
  int rc;
  // E[a,s,c] = sum C[a,i] T[i,s,k] C[k,c]
  rc = stage_reduced_corner(h, h->C, h->T, h->W); if (rc) return rc;
  { GemmCall c{h->W, chi, 0, h->C, chi, h->E, plain_map(chi), IndexMap{1, 1, 0}, (int)m, chi, chi, 0}; GEMM(h, c); }
  // Z4 = tr C^4 = tr (C2 C2)
  { GemmCall c{h->C, chi, 0, h->C, chi, h->Wc, plain_map(chi), IndexMap{1, 1, 0}, chi, chi, chi, 0}; GEMM(h, c); }
  trace_prod_partial_kernel<<<148, 256, 0, h->stream>>>(h->Wc, chi, h->partial + 2 * kPartialBlocks);
  sum_partial_kernel<<<1, 256, 0, h->stream>>>(h->partial + 2 * kPartialBlocks, 148, h->scal + 2);
  h->launches += 2;
  // Z2 = sum E^2
  rc = reduce_dot(h, h->E, h->E, m * chi, h->scal + 3); if (rc) return rc;
  // Z1 = sum E[a,u,c] T[a,l,a'] a[u,l,d,r] T[c,r,c'] E[a',d,c']
  rc = stage_half_absorb(h, h->E, h->T, h->P); if (rc) return rc;          // F[u,l,c,a']
  rc = stage_absorb_a(h, h->P, h->S, 1); if (rc) return rc;                // G~[c,r,a',d]
  { GemmCall c{h->S, m, 1, h->T, chi, h->W, plain_map(chi), IndexMap{1, 1, 0}, (int)m, chi, (int)m, 0}; GEMM(h, c); }
  rc = reduce_dot(h, h->W, h->E, m * chi, h->scal + 4); if (rc) return rc; // H[(a',d),c'] . E
  CU(h, cudaMemcpyAsync(h->h_pinned + 2, h->scal + 2, 3 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  double Z4 = h->h_pinned[2], Z2 = h->h_pinned[3], Z1 = h->h_pinned[4];
  *kappa = Z1 * Z4 / (Z2 * Z2);
  return QRCTM_OK;
}

int qrctm_energy_nn(qrctm_t* h, const double* H, double* e_bond, double* rho_out) {
  if (!h || !H || !e_bond) return h ? fail(h, QRCTM_ERR_INVALID_ARG, "null argument") : QRCTM_ERR_INVALID_ARG;
  if (!h->have_A || !h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "set_A and set_env first");
  const int d = h->d, chi = h->chi;
  if (d > 4) return fail(h, QRCTM_ERR_INVALID_ARG, "qrctm_energy_nn supports d <= 4");
  if (is_device_ptr(H) || (rho_out && is_device_ptr(rho_out))) return fail(h, QRCTM_ERR_INVALID_ARG, "H, rho: host pointers");
  const long long m = h->m, nlh = m * chi;
  int rc;
  // half network LH^{ss'} = (E3) with c~ for Q and a^{ss'} for a
  rc = stage_reduced_corner(h, h->C, h->T, h->X); if (rc) return rc;
  rc = stage_half_absorb(h, h->X, h->T, h->P); if (rc) return rc;
  const long long b2 = (long long)h->b * h->b, n = b2 * b2;
  int nb = (int)((n + 255) / 256); if (nb > 148 * 8) nb = 148 * 8;
  for (int s = 0; s < d; ++s)
    for (int sp = 0; sp < d; ++sp) {
      build_a_pair_kernel<<<nb, 256, 0, h->stream>>>(h->A, h->D, s, sp, h->a2_mat, h->L.lda_a);
      h->launches += 1;
      rc = stage_absorb_a(h, h->P, h->S, 0, h->a2_mat); if (rc) return rc;
      rc = stage_project(h, h->S, h->X, h->LH + (size_t)(s * d + sp) * nlh); if (rc) return rc;
    }
  // rho[s1,s1',s2,s2'] = <LH^{s1s1'}, LH^{s2s2'}>   (symmetric under exchange of the two pairs)
  const int d2 = d * d;
  for (int p = 0; p < d2; ++p)
    for (int q = p; q < d2; ++q) {
      rc = reduce_dot(h, h->LH + (size_t)p * nlh, h->LH + (size_t)q * nlh, nlh, h->rho + p * d2 + q); if (rc) return rc;
    }
  CU(h, cudaMemcpyAsync(h->h_pinned + 64, h->rho, sizeof(double) * d2 * d2, cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  const double* r = h->h_pinned + 64;
  double num = 0.0, den = 0.0;
  for (int s1 = 0; s1 < d; ++s1) for (int s1p = 0; s1p < d; ++s1p)
    for (int s2 = 0; s2 < d; ++s2) for (int s2p = 0; s2p < d; ++s2p) {
      const int p = s1 * d + s1p, q = s2 * d + s2p;
      const double v = p <= q ? r[p * d2 + q] : r[q * d2 + p];
      if (rho_out) rho_out[((s1 * d + s1p) * d + s2) * d + s2p] = v;
      num += v * H[(size_t)(s1 * d + s2) * d2 + (s1p * d + s2p)];
      if (s1 == s1p && s2 == s2p) den += v;
    }
  if (!(den != 0.0)) return fail(h, QRCTM_ERR_NUMERIC, "zero two-site norm");
  *e_bond = num / den;
  return QRCTM_OK;
}

int qrctm_r_diag_ratio(qrctm_t* h, double* ratio) {
  if (!h || !ratio) return QRCTM_ERR_INVALID_ARG;
  r_diag_minmax_kernel<<<1, 256, 0, h->stream>>>(h->R, h->chi, h->scal + 5);
  h->launches += 1;
  CU(h, cudaMemcpyAsync(h->h_pinned + 5, h->scal + 5, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  *ratio = h->h_pinned[6] != 0.0 ? h->h_pinned[5] / h->h_pinned[6] : 0.0;
  return QRCTM_OK;
}

int qrctm_profile_step(qrctm_t* h, float* ms) {
  if (!h || !ms) return QRCTM_ERR_INVALID_ARG;
  if (!h->have_A || !h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "set_A and set_env first");
  cudaEvent_t ev[QRCTM_NSTAGE + 1];
  for (int i = 0; i <= QRCTM_NSTAGE; ++i) CU(h, cudaEventCreate(&ev[i]));
  int rc = do_step(h, ev);
  cudaError_t e = cudaStreamSynchronize(h->stream);
  if (rc == QRCTM_OK && e == cudaSuccess)
    for (int i = 0; i < QRCTM_NSTAGE; ++i) cudaEventElapsedTime(&ms[i], ev[i], ev[i + 1]);
  for (int i = 0; i <= QRCTM_NSTAGE; ++i) cudaEventDestroy(ev[i]);
  if (rc) return rc;
  CU(h, e);
  return QRCTM_OK;
}

int qrctm_gemm_f64(void* cuda_stream, int path, int transA, int M, int N, int K, const double* A, long long lda,
                   const double* B, long long ldb, double* Cmat, long long ldc) {
  if (!A || !B || !Cmat || M < 0 || N < 0 || K < 0 || (path != 0 && path != 1)) return QRCTM_ERR_INVALID_ARG;
  GemmCall c{A, lda, transA ? 1 : 0, B, ldb, Cmat, plain_map(ldc), IndexMap{1, 1, 0}, M, N, K, 0};
  cudaError_t e;
  int nl = launch_gemm(static_cast<cudaStream_t>(cuda_stream), path, c, nullptr, 0, &e);
  return nl < 0 ? QRCTM_ERR_CUDA : QRCTM_OK;
}

unsigned long long qrctm_qr_work_bytes(int rows, int cols) { return qr_work_bytes_impl(rows, cols); }

int qrctm_qr_f64(void* cuda_stream, int path, int rows, int cols, const double* X, double* Q, double* R,
                 void* work) {
  if (!X || !Q || !R || !work || rows < 1 || cols < 1 || cols > rows || path < 0 || path > 2)
    return QRCTM_ERR_INVALID_ARG;
  cudaError_t e;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  long long nl = path != 1 ? qr_factor_blocked(st, path, rows, cols, X, Q, R, work, &e)
                           : qr_factor_level2(st, rows, cols, X, Q, R, work, &e);
  return nl < 0 ? QRCTM_ERR_CUDA : QRCTM_OK;
}

int qrctm_probe_fp64(int kind, int iters, double* tflops) {
  if (!tflops || iters < 1 || (kind != 0 && kind != 1)) return QRCTM_ERR_INVALID_ARG;
  cudaDeviceProp p;
  if (cudaGetDeviceProperties(&p, 0) != cudaSuccess) { cudaGetLastError(); return QRCTM_ERR_CUDA; }
  const int blocks = p.multiProcessorCount * 2, threads = 256;
  double* out = nullptr;
  if (cudaMalloc(&out, sizeof(double) * blocks * threads) != cudaSuccess) { cudaGetLastError(); return QRCTM_ERR_CUDA; }
  cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
  auto go = [&] {
    if (kind == 0) probe_dfma_kernel<<<blocks, threads>>>(out, iters, 1e-3);
    else probe_dmma_kernel<<<blocks, threads>>>(out, iters, 1e-3);
  };
  go(); cudaDeviceSynchronize();
  cudaEventRecord(a); go(); cudaEventRecord(b); cudaEventSynchronize(b);
  float ms = 0; cudaEventElapsedTime(&ms, a, b);
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(out);
  if (cudaGetLastError() != cudaSuccess || ms <= 0) return QRCTM_ERR_CUDA;
  double nthr = (double)blocks * threads;
  double flops = kind == 0 ? nthr * iters * 16.0 * 2.0 : (nthr / 32.0) * iters * 8.0 * 512.0;
  *tflops = flops / (ms * 1e-3) / 1e12;
  return QRCTM_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ NEXT-2: initialisation and eigen step
namespace {

// K1, K3, K4 with C, T themselves give C~; its chi_new largest-|lambda| eigenpairs give U (for Q) and
// C' = diag(lambda); T' = (E3) with U for Q  (Fig. 1(d)).
int stage_eig_step(qrctm* h, int chi_new) {
  const long long mi = h->m;
  const size_t need = eigh_work_bytes_impl(mi, chi_new) + sizeof(double) * (size_t)chi_new + 256;
  if (h->eigwork_bytes < need) {
    CU(h, cudaStreamSynchronize(h->stream));
    if (h->eigwork) { cudaFree(h->eigwork); h->eigwork = nullptr; h->eigwork_bytes = 0; }
    CU(h, cudaMalloc(&h->eigwork, need));
    h->eigwork_bytes = need;
  }
  double* lam = static_cast<double*>(h->eigwork);
  void* work = static_cast<char*>(h->eigwork) + align_up(sizeof(double) * (size_t)chi_new);
  nvtxRangePushA("E1_enlarged_corner");
  int rc = stage_reduced_corner(h, h->C, h->T, h->X);
  if (!rc) rc = stage_half_absorb(h, h->X, h->T, h->P);
  if (!rc) rc = stage_absorb_a(h, h->P, h->S, 0);                        // S = C~[(J,d),(k,r)]
  nvtxRangePop();
  if (rc) return rc;
  symmetrize_inplace_kernel<<<592, 256, 0, h->stream>>>(h->S, (int)mi);
  h->launches += 1;
  nvtxRangePushA("E2_eigh");
  cudaError_t e;
  long long nl = eigh_top(h->stream, (int)mi, chi_new, h->S, lam, h->Q, work, &e);
  nvtxRangePop();
  if (nl < 0) return fail(h, QRCTM_ERR_CUDA, "eigh", e);
  h->launches += nl;
  nvtxRangePushA("E3_edge");
  rc = stage_half_absorb(h, h->Q, h->T, h->P, chi_new);
  if (!rc) rc = stage_absorb_a(h, h->P, h->S, 0, nullptr, chi_new);
  if (!rc) rc = stage_project(h, h->S, h->Q, h->Tn, chi_new);
  nvtxRangePop();
  if (rc) return rc;
  diag_matrix_kernel<<<(chi_new * chi_new + 255) / 256, 256, 0, h->stream>>>(lam, chi_new, h->Cn);
  h->launches += 1;
  CU(h, cudaGetLastError());
  h->eig_rows = (int)mi; h->eig_cols = chi_new;
  set_chi(h, chi_new);
  return stage_normalize(h, h->Cn, h->Tn);
}

}  // namespace

extern "C" {

int qrctm_get_chi(const qrctm_t* h, int* chi, int* chi_capacity) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (chi) *chi = h->chi;
  if (chi_capacity) *chi_capacity = h->chi_cap;
  return QRCTM_OK;
}

int qrctm_init_bulk(qrctm_t* h) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (!h->have_A) return fail(h, QRCTM_ERR_NOT_READY, "set_A first");
  if (h->b > h->chi_cap) return fail(h, QRCTM_ERR_INVALID_ARG, "bulk initialisation needs D^2 <= chi");
  CU(h, cudaStreamSynchronize(h->stream));
  set_chi(h, h->b);
  const long long tot = (long long)h->b * h->b * (1 + h->b);
  int nb = (int)((tot + 255) / 256); if (nb > 1184) nb = 1184;
  bulk_init_kernel<<<nb, 256, 0, h->stream>>>(h->A, h->d, h->D, h->Cn, h->Tn);
  h->launches += 1;
  CU(h, cudaGetLastError());
  CU(h, cudaMemsetAsync(h->flag, 0, sizeof(int), h->stream));
  int rc = stage_normalize(h, h->Cn, h->Tn); if (rc) return rc;
  rc = check_flag(h); if (rc) return rc;
  CU(h, cudaMemsetAsync(h->s_prev, 0, sizeof(double) * h->chi_cap, h->stream));
  h->need_s0 = 1;
  h->have_env = true;
  return QRCTM_OK;
}

int qrctm_eig_step(qrctm_t* h, int chi_new) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (!h->have_A || !h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "set_A and set_env / init_bulk first");
  if (chi_new == 0) chi_new = h->chi;
  if (chi_new < 1 || chi_new > h->chi_cap || chi_new > h->m) return fail(h, QRCTM_ERR_INVALID_ARG, "chi_new out of range");
  if (h->m > EIGH_MAX_N) return fail(h, QRCTM_ERR_INVALID_ARG, "eigen step supports chi*D^2 <= 14000");
  int rc = stage_eig_step(h, chi_new); if (rc) return rc;
  rc = check_flag(h); if (rc) return rc;
  CU(h, cudaMemsetAsync(h->s_prev, 0, sizeof(double) * h->chi_cap, h->stream));
  h->need_s0 = 1;
  return QRCTM_OK;
}

int qrctm_get_eig(qrctm_t* h, double* U, double* lam, int* rows, int* cols) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (!h->eig_rows || !h->eigwork) return fail(h, QRCTM_ERR_NOT_READY, "no eigen step yet");
  if (rows) *rows = h->eig_rows;
  if (cols) *cols = h->eig_cols;
  if (U) CU(h, copy_out(U, h->Q, (size_t)h->eig_rows * h->eig_cols, h->stream));
  if (lam) CU(h, copy_out(lam, static_cast<double*>(h->eigwork), (size_t)h->eig_cols, h->stream));
  return QRCTM_OK;
}

int qrctm_warmup(qrctm_t* h, int n_eig_steps) {
  if (!h || n_eig_steps < 0) return h ? fail(h, QRCTM_ERR_INVALID_ARG, "n_eig_steps < 0") : QRCTM_ERR_INVALID_ARG;
  int rc = qrctm_init_bulk(h); if (rc) return rc;
  for (int i = 0; i < n_eig_steps; ++i) {
    long long grown = h->m;                                   // chi * D^2
    int chi_new = grown > h->chi_cap ? h->chi_cap : (int)grown;
    rc = qrctm_eig_step(h, chi_new); if (rc) return rc;
  }
  return QRCTM_OK;
}

unsigned long long qrctm_eigh_work_bytes(int n, int k) { return eigh_work_bytes_impl(n, k); }

int qrctm_eigh_top_f64(void* cuda_stream, int n, int k, double* A, double* lam, double* U, void* work) {
  if (!A || !lam || !U || !work || n < 1 || k < 1 || k > n || n > EIGH_MAX_N) return QRCTM_ERR_INVALID_ARG;
  cudaError_t e;
  long long nl = eigh_top(static_cast<cudaStream_t>(cuda_stream), n, k, A, lam, U, work, &e);
  return nl < 0 ? QRCTM_ERR_CUDA : QRCTM_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ NEXT-4: one iteration sharded over the column index m of Q
namespace {

void shard_range(int chi, int rank, int nranks, int* m0, int* m1) {      // contiguous, sizes differ by at most one
  const int q = chi / nranks, r = chi % nranks;
  *m0 = rank * q + (rank < r ? rank : r);
  *m1 = *m0 + q + (rank < r ? 1 : 0);
}

}  // namespace

extern "C" {

int qrctm_shard_range(int chi, int rank, int nranks, int* m0, int* m1) {
  if (chi < 1 || nranks < 1 || rank < 0 || rank >= nranks || !m0 || !m1) return QRCTM_ERR_INVALID_ARG;
  shard_range(chi, rank, nranks, m0, m1);
  return QRCTM_OK;
}

int qrctm_shard_front(qrctm_t* h, int rank, int nranks) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (!h->have_A || !h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "set_A and set_env first");
  if (nranks < 1 || rank < 0 || rank >= nranks) return fail(h, QRCTM_ERR_INVALID_ARG, "rank / nranks");
  h->eig_rows = 0;
  const int chi = h->chi, b = h->b; const long long m = h->m, bc = (long long)b * chi;
  int m0, m1; shard_range(chi, rank, nranks, &m0, &m1);
  const int co = m1 - m0;
  // replicated: K1, K2 (0.3 % of the flops)
  int rc = stage_reduced_corner(h, h->C, h->T, h->X); if (rc) return rc;
  cudaError_t e;
  long long nl = h->qr_path != 1 ? qr_factor_blocked(h->stream, h->qr_path, m, chi, h->X, h->Q, h->R, h->qrwork, &e)
                                 : qr_factor_level2(h->stream, m, chi, h->X, h->Q, h->R, h->qrwork, &e);
  if (nl < 0) return fail(h, QRCTM_ERR_CUDA, "qr", e);
  h->launches += nl;
  // the other ranks' rows of T' and the partial C' start from zero, so that either an all-gather of the slices or a
  // plain sum over ranks assembles the full tensors
  CU(h, cudaMemsetAsync(h->Tn, 0, sizeof(double) * m * chi, h->stream));
  CU(h, cudaMemsetAsync(h->Cn, 0, sizeof(double) * chi * chi, h->stream));
  if (co == 0) return QRCTM_OK;
  // this rank's slice: K3, K4, K5 with the columns [m0, m1) of Q in place of Q on the open leg
  slice_cols_kernel<<<296, 256, 0, h->stream>>>(h->Q, m, chi, m0, co, h->E);
  transpose_rows_kernel<<<(chi * co + 255) / 256, 256, 0, h->stream>>>(h->R, chi, m0, co, h->Rt);
  h->launches += 2;
  CU(h, cudaGetLastError());
  rc = stage_half_absorb(h, h->E, h->T, h->P, co); if (rc) return rc;
  rc = stage_absorb_a(h, h->P, h->S, 0, nullptr, co); if (rc) return rc;
  double* Tn_slice = h->Tn + (long long)m0 * bc;                       // rows (m, r), m in [m0, m1)
  rc = stage_project(h, h->S, h->Q, Tn_slice, co, chi); if (rc) return rc;
  // partial (E4): W[(mo,r),n] = sum_k R[m0+mo,k] Q[k,(r,n)];  C'_part[p,n] = sum_{(mo,r)} T'[(mo,r),p] W[(mo,r),n]
  GemmCall c1{h->Q, bc, 1, h->Rt, co, h->W, IndexMap{1, 1, 0}, plain_map(bc), (int)bc, co, chi, 0};
  GEMM(h, c1);
  GemmCall c2{Tn_slice, chi, 1, h->W, chi, h->Cn, plain_map(chi), IndexMap{1, 1, 0}, chi, chi, co * b, 0};
  GEMM(h, c2);
  return QRCTM_OK;
}

int qrctm_shard_buffers(qrctm_t* h, double** Cn, double** Tn) {
  if (!h || !Cn || !Tn) return QRCTM_ERR_INVALID_ARG;
  *Cn = h->Cn; *Tn = h->Tn;
  return QRCTM_OK;
}

int qrctm_shard_finish(qrctm_t* h) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (!h->have_A || !h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "set_A and set_env first");
  return stage_normalize(h, h->Cn, h->Tn);
}

}  // extern "C"
