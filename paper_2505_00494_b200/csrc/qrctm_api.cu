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
#include "cholqr.cuh"
#include "small_step.cuh"
#include "spectrum.cuh"
#include "eigh.cuh"

using namespace qk;

namespace {

constexpr int kPartialBlocks = 592;   // 4 x 148 blocks for the reduction kernels
// pinned host scratch (doubles): [0] delta, [2..6] scalars read back by the observables, [32..] the NaN/zero flag
// (as int), [kPinRho .. kPinRho + kRhoMax) the two-site RDM of qrctm_energy_nn (d <= kEnergyMaxD)
constexpr int kPinFlag = 32, kPinRho = 64, kEnergyMaxD = 4;
constexpr int kRhoMax = kEnergyMaxD * kEnergyMaxD * kEnergyMaxD * kEnergyMaxD;
constexpr int kPinDoubles = kPinRho + kRhoMax;
constexpr size_t kAlign = 256;

inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct Layout {   // byte offsets into the workspace
  size_t A, a_mat, a2_mat, LH, rho, B1, B2, P1, C, T, Cn, Tn, X, Q, R, Rt, P, S, W, E, splitk, partial, scal, flag, hist, Wc, dvec, evec,
      vv, pv, eig, s, s_prev, s_tmp, delta, qrwork, k8work, total;
  long long lda_a, ld1, ld2;
  size_t splitk_elems, qrwork_bytes, k8work_bytes;
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
  int k8_old;             // 1: K8 on the round-1 tridiagonalisation kernel (QRCTM_OPT_K8_PATH, for cross-checks)
  int small_off;          // 1: never use the whole-iteration kernels for tiny problems (QRCTM_OPT_SMALL_PATH)
  int small_force;        // 1: use them whenever the working set fits (QRCTM_OPT_SMALL_PATH = 2), not only for chi <= 8
  int small_smem;         // opt-in shared memory available to them (0: not queried yet, -1: unavailable)
  long long launches;
  cudaEvent_t ev[QRCTM_NSTAGE + 2];
  bool have_ev;
  cudaGraphExec_t g_front, g_k7;  // captured K1..K6 and K7 (replayed by step/run)
  cudaGraphExec_t g_qrfb;         // {set condition; IF -> Householder QR}: the device-decided fallback of K2 for direct launches
  long long g_front_n, g_k7_n;    // kernels per replay
  int use_graph, warm_steps, graph_failed;
  int need_s0;                    // spectrum of the environment set by set_env not computed yet (lazy)
  cudaStream_t cap_aux;         // captures the body of the conditional Householder fallback of K2 (never runs work itself)
  cudaStream_t branch;          // K6's first product W = R.Q (needs only K2's outputs) runs here beside K3..K5
  cudaEvent_t ev_fork, ev_join;
  cudaStream_t side;            // high-priority stream for the overlapped convergence check
  cudaEvent_t ev_env, ev_spec;  // environment ready (main) / spectrum done (side)
  int overlap;
  double stage_ms[QRCTM_NSTAGE + 1];
  long long stage_steps;
  char err[256];
  double* h_pinned;       // [0] delta, [1..] scratch ; pinned host
  int* h_flag;
  // typed views
  double *A, *a_mat, *a2_mat, *LH, *rho, *B1, *B2, *P1, *C, *T, *Cn, *Tn, *X, *Q, *R, *Rt, *P, *S, *W, *E, *splitk, *partial, *scal, *hist, *Wc,
      *dvec, *evec, *vv, *pv, *eig, *s, *s_prev, *s_tmp, *delta;
  int* flag;
  void* qrwork;
  void* k8work;                 // scratch of K8's multi-CTA tridiagonalisation (chi too large for one SM), or null
};

namespace {

unsigned long long qr_work_bytes_impl(long long rows, int cols);
struct EighWork;
size_t eigh_layout(long long n, int k, char* base, EighWork* w);
constexpr int kMaxChi = 800;            // form-Q back substitution keeps chi/16 blocks of 4 KB in shared memory
constexpr int kK8SmemMaxChi = 200;      // above this chi a scratch area for the multi-CTA tridiagonalisation is carved

bool make_layout(int d, int D, int chi, Layout* L) {
  if (d < 1 || D < 1 || chi < 1) return false;
  if (D > 32 || chi > kMaxChi || d > 64) return false;               // sizes this build supports
  long long b = (long long)D * D, m = b * chi;
  long long b2 = b * b;
  L->lda_a = (b2 + 15) / 16 * 16;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
  const size_t dbl = sizeof(double);
  L->A = take(dbl * d * b2);
  L->a_mat = take(dbl * b2 * L->lda_a);
  L->a2_mat = take(dbl * b2 * L->lda_a);
  L->LH = take(d <= kEnergyMaxD ? dbl * (size_t)d * d * m * chi : 0);
  L->rho = take(dbl * kRhoMax);
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
  L->flag = take(sizeof(int) * 4);          // [0] NaN/zero-norm flag, [1] number of history records written
  L->hist = take(dbl * 4 * QRCTM_HIST_CAP);
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
  L->k8work_bytes = chi > kK8SmemMaxChi ? eigh_layout(chi, 1, nullptr, nullptr) : 0;
  L->k8work = take(L->k8work_bytes);
  L->total = off;
  return true;
}

void bind_views(qrctm* h) {
  char* B = h->base;
  const Layout& L = h->L;
#define V_(name) h->name = reinterpret_cast<double*>(B + L.name)
  V_(A); V_(a_mat); V_(a2_mat); V_(LH); V_(rho); V_(B1); V_(B2); V_(P1); V_(C); V_(T); V_(Cn); V_(Tn); V_(X); V_(Q); V_(R); V_(Rt); V_(P); V_(S); V_(W);
  V_(E); V_(splitk); V_(partial); V_(scal); V_(hist); V_(Wc); V_(dvec); V_(evec); V_(vv); V_(pv); V_(eig); V_(s);
  V_(s_prev); V_(s_tmp); V_(delta);
#undef V_
  h->flag = reinterpret_cast<int*>(B + L.flag);
  h->qrwork = B + L.qrwork;
  h->k8work = L.k8work_bytes ? B + L.k8work : nullptr;
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

#include "gemm_launch.cuh"

}  // namespace

namespace {

#include "qr_driver.cuh"
#include "eigh_driver.cuh"

}  // namespace

// ------------------------------------------------------------------ step stages
namespace {

#include "stages.cuh"

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
  {   // one device per process (the one-time kernel attributes are cached per process): fail loudly on a second one
    static int first_device = -1;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return QRCTM_ERR_CUDA; }
    if (first_device < 0) first_device = dev;
    else if (dev != first_device) return QRCTM_ERR_INVALID_ARG;
  }
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
  if (cudaMallocHost(&hp, kPinDoubles * sizeof(double)) != cudaSuccess) {
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
  if (cudaStreamCreateWithFlags(&h->cap_aux, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); h->cap_aux = nullptr; }
  if (cudaStreamCreateWithFlags(&h->branch, cudaStreamNonBlocking) != cudaSuccess ||
      cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); h->branch = nullptr; }
  h->h_flag = reinterpret_cast<int*>(h->h_pinned + kPinFlag);
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
  if (h->cap_aux) cudaStreamDestroy(h->cap_aux);
  if (h->branch) { cudaStreamSynchronize(h->branch); cudaStreamDestroy(h->branch); cudaEventDestroy(h->ev_fork); cudaEventDestroy(h->ev_join); }
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
  CU(h, cudaMemsetAsync(h->flag, 0, 2 * sizeof(int), h->stream));      // numeric flag and the history counter
  int rc = stage_normalize(h, h->Cn, h->Tn); if (rc) return rc;
  rc = check_flag(h); if (rc) return rc;
  CU(h, cudaMemsetAsync(h->s_prev, 0, sizeof(double) * h->chi, h->stream));
  h->need_s0 = 1;      // s_prev = spectrum(C0) is computed by the next qrctm_run, overlapped with its first step
  h->have_env = true;
  return QRCTM_OK;
}

// The convergence history of a freshly set environment starts at s_prev = spectrum(C0).  qrctm_run computes it lazily
// (under its first step); every other entry that is about to overwrite C computes it first.
static int ensure_s0(qrctm* h) {
  if (!h->need_s0) return QRCTM_OK;
  int rc = stage_spectrum(h, h->s, 1, h->stream); if (rc) return rc;
  h->need_s0 = 0;
  return QRCTM_OK;
}

int qrctm_step(qrctm_t* h) {
  if (!h) return QRCTM_ERR_INVALID_ARG;
  if (!h->have_A || !h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "set_A and set_env first");
  { int rc0 = ensure_s0(h); if (rc0) return rc0; }
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
  if (max_iter > 0 && h->check_every >= 2 && !h->time_stages && !h->k8_old && h->chi <= SPEC_FUSED_MAX_N && small_ok(h)) {
    // tiny problem, spectrum not wanted after every step: the whole loop in one launch, convergence decided on the
    // device (small_step.cuh).  With CHECK_EVERY = 1 the pipelined driver below is faster: there K8 of step k runs on
    // the side stream under step k+1, here the one CTA does them one after the other (measured at cfg0: 46 us per
    // step against 51)
    static bool attr = false;
    if (!attr) {
      CU(h, cudaFuncSetAttribute(small_run_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, h->small_smem - 2048));
      attr = true;                                              // (2 KB: the kernel's static shared memory)
    }
    const size_t smem = small_run_smem_bytes(h->b, h->chi);
    if (smem + 2048 <= (size_t)h->small_smem) {
      small_run_kernel<<<1, SMALL_NT, smem, h->stream>>>(h->C, h->T, h->a_mat, h->L.lda_a, h->b, h->chi, h->symmetrize, h->X,
                                                         h->Q, h->R, h->Tn, h->Cn, h->scal, h->flag, h->hist, h->flag + 1, h->eig,
                                                         h->s, h->s_prev, h->delta, h->need_s0, max_iter, tol, h->check_every,
                                                         h->scal + 10);
      h->launches += 1;
      h->need_s0 = 0;
      CU(h, cudaGetLastError());
      CU(h, cudaMemcpyAsync(h->h_pinned + 10, h->scal + 10, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
      int rcf = check_flag(h); if (rcf) return rcf;             // synchronises
      if (iters_done) *iters_done = (int)h->h_pinned[10];
      if (final_delta) *final_delta = h->h_pinned[11];
      h->warm_steps += 1;
      return QRCTM_OK;
    }
  }
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
        bool wrote = false;
        rc = stage_spectrum(h, h->s, 1, h->side, true, &wrote); if (rc) return rc;
        if (!wrote) {       // paths whose last kernel does not write the mapped host words itself
          CU(h, cudaMemcpyAsync(h->h_pinned, h->delta, sizeof(double), cudaMemcpyDeviceToHost, h->side));
          CU(h, cudaMemcpyAsync(h->h_flag, h->flag, sizeof(int), cudaMemcpyDeviceToHost, h->side));
        }
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
    case QRCTM_OPT_QR_PATH:     if (value < 0 || value > 4) break; h->qr_path = value; return QRCTM_OK;
    case QRCTM_OPT_OVERLAP_CHECK: if (value != 0 && value != 1) break; h->overlap = value; return QRCTM_OK;
    case QRCTM_OPT_ABSORB_MODE: if (value < 0 || value > 2) break; h->absorb_mode = value; return QRCTM_OK;
    case QRCTM_OPT_USE_GRAPH:   if (value != 0 && value != 1) break; h->use_graph = value; return QRCTM_OK;
    case QRCTM_OPT_TIME_STAGES: if (value != 0 && value != 1) break; h->time_stages = value; return QRCTM_OK;
    case QRCTM_OPT_K8_PATH:     if (value != 0 && value != 1) break; h->k8_old = value; return QRCTM_OK;
    case QRCTM_OPT_SMALL_PATH:  if (value < 0 || value > 2) break; h->small_off = value == 1; h->small_force = value == 2; return QRCTM_OK;
    default: break;
  }
  return fail(h, QRCTM_ERR_INVALID_ARG, "bad option key/value");
}

long long qrctm_launch_count(const qrctm_t* h) { return h ? h->launches : 0; }

int qrctm_get_history(qrctm_t* h, double* out, int max_records, int* n_steps) {
  if (!h || !n_steps || max_records < 0 || (max_records > 0 && !out)) return h ? fail(h, QRCTM_ERR_INVALID_ARG, "bad argument") : QRCTM_ERR_INVALID_ARG;
  if (out && is_device_ptr(out)) return fail(h, QRCTM_ERR_INVALID_ARG, "history: host pointer");
  if (h->side) CU(h, cudaStreamSynchronize(h->side));
  int n = 0;
  CU(h, cudaMemcpyAsync(&n, h->flag + 1, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  *n_steps = n;
  int take = n < max_records ? n : max_records;
  if (take > QRCTM_HIST_CAP) take = QRCTM_HIST_CAP;
  for (int r = 0; r < take; ++r) {          // chronological: the last `take` records
    const int idx = (n - take + r) % QRCTM_HIST_CAP;
    CU(h, cudaMemcpyAsync(out + 4 * (size_t)r, h->hist + 4 * (size_t)idx, 4 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  }
  CU(h, cudaStreamSynchronize(h->stream));
  return QRCTM_OK;
}

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
  static_assert(kPinRho + kRhoMax <= kPinDoubles, "pinned RDM area");
  if (d > kEnergyMaxD) return fail(h, QRCTM_ERR_INVALID_ARG, "qrctm_energy_nn supports d <= 4");
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
  CU(h, cudaMemcpyAsync(h->h_pinned + kPinRho, h->rho, sizeof(double) * d2 * d2, cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  const double* r = h->h_pinned + kPinRho;
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

int qrctm_edge_update(qrctm_t* h, const double* U, int ncols, double* Tout) {
  if (!h || !U || !Tout) return h ? fail(h, QRCTM_ERR_INVALID_ARG, "null argument") : QRCTM_ERR_INVALID_ARG;
  if (!h->have_A || !h->have_env) return fail(h, QRCTM_ERR_NOT_READY, "set_A and set_env first");
  if (ncols < 1 || ncols > h->chi_cap) return fail(h, QRCTM_ERR_INVALID_ARG, "ncols out of range");
  const long long mo = (long long)ncols * h->b;
  CU(h, copy_in(h->E, U, (size_t)h->m * ncols, h->stream));
  int rc = stage_half_absorb(h, h->E, h->T, h->P, ncols); if (rc) return rc;
  rc = stage_absorb_a(h, h->P, h->S, 0, nullptr, ncols); if (rc) return rc;
  rc = stage_project(h, h->S, h->E, h->W, ncols); if (rc) return rc;
  CU(h, copy_out(Tout, h->W, (size_t)mo * ncols, h->stream));
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
  { int rc0 = ensure_s0(h); if (rc0) return rc0; }
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

int qrctm_gemm_f64_ws(void* cuda_stream, int path, int transA, int M, int N, int K, const double* A, long long lda,
                      const double* B, long long ldb, double* Cmat, long long ldc, void* work,
                      unsigned long long work_bytes) {
  if (!A || !B || !Cmat || M < 0 || N < 0 || K < 0 || (path != 0 && path != 1)) return QRCTM_ERR_INVALID_ARG;
  if ((work == nullptr && work_bytes != 0) || (reinterpret_cast<uintptr_t>(work) & 15)) return QRCTM_ERR_INVALID_ARG;
  GemmCall c{A, lda, transA ? 1 : 0, B, ldb, Cmat, plain_map(ldc), IndexMap{1, 1, 0}, M, N, K, 0};
  cudaError_t e;
  int nl = launch_gemm(static_cast<cudaStream_t>(cuda_stream), path, c, static_cast<double*>(work),
                       (size_t)(work_bytes / sizeof(double)), &e);
  return nl < 0 ? QRCTM_ERR_CUDA : QRCTM_OK;
}

}  // extern "C"

// ---- allocation-free GEMM entry: the K-splitting scratch lives in a file-scope device array (16 MiB on every GPU that
// loads the library, until exit).  In host code `g_noalloc_scratch` is only a stand-in for the symbol: the device
// address is looked up once per device with cudaGetSymbolAddress and that pointer is what the kernels get.
namespace {
constexpr size_t kNoAllocElems = (size_t)1 << 21;                 // 2 Mi doubles = 16 MiB
constexpr long long kNoAllocMaxMN = 65536;                        // M * N of one call (32 K-splits of it fit the array)
constexpr int kNoAllocMaxDev = 64;
}  // namespace
static __device__ __align__(256) double g_noalloc_scratch[kNoAllocElems];
namespace {
double* g_noalloc_ptr[kNoAllocMaxDev];                            // per device, filled on first use
thread_local char g_noalloc_err[200] = "";
int noalloc_fail(int code, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess) snprintf(g_noalloc_err, sizeof(g_noalloc_err), "%s: %s", what, cudaGetErrorString(e));
  else snprintf(g_noalloc_err, sizeof(g_noalloc_err), "%s", what);
  return code;
}
}  // namespace

extern "C" {

const char* qrctm_noalloc_last_error(void) { return g_noalloc_err; }

int qrctm_gemm_f64_noalloc(void* cuda_stream, int transA, int M, int N, int K, const double* A, long long lda,
                           const double* B, long long ldb, double* Cmat, long long ldc) {
  g_noalloc_err[0] = 0;
  if (!A || !B || !Cmat || M < 1 || N < 1 || K < 1) return noalloc_fail(QRCTM_ERR_INVALID_ARG, "null pointer or empty shape");
  if ((long long)M * N > kNoAllocMaxMN)
    return noalloc_fail(QRCTM_ERR_INVALID_ARG, "qrctm_gemm_f64_noalloc: M * N exceeds 65536 (the static scratch holds 32 K-splits of a 65536-element output); use qrctm_gemm_f64_ws");
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { cudaGetLastError(); return noalloc_fail(QRCTM_ERR_CUDA, "cudaGetDevice", e); }
  if (dev < 0 || dev >= kNoAllocMaxDev) return noalloc_fail(QRCTM_ERR_INVALID_ARG, "device index beyond 63");
  if (!g_noalloc_ptr[dev]) {                                      // once per device, with that device current
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p) { cudaGetLastError(); return noalloc_fail(QRCTM_ERR_CUDA, "cudaGetSymbolAddress(g_noalloc_scratch)", e); }
    g_noalloc_ptr[dev] = p;
  }
  GemmCall c{A, lda, transA ? 1 : 0, B, ldb, Cmat, plain_map(ldc), IndexMap{1, 1, 0}, M, N, K, 0};
  int nl = launch_gemm(static_cast<cudaStream_t>(cuda_stream), 0, c, g_noalloc_ptr[dev], kNoAllocElems, &e);
  if (nl < 0) return noalloc_fail(QRCTM_ERR_CUDA, "gemm launch", e);
  return QRCTM_OK;
}

unsigned long long qrctm_qr_work_bytes(int rows, int cols) { return qr_work_bytes_impl(rows, cols); }

int qrctm_qr_f64(void* cuda_stream, int path, int rows, int cols, const double* X, double* Q, double* R,
                 void* work) {
  if (!X || !Q || !R || !work || rows < 1 || cols < 1 || cols > rows || cols > kMaxChi || path < 0 || path > 4)
    return QRCTM_ERR_INVALID_ARG;
  cudaError_t e;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  long long nl = path != 1 ? qr_factor_blocked(st, path, rows, cols, X, Q, R, work, &e)
                           : qr_factor_level2(st, rows, cols, X, Q, R, work, &e);
  return nl < 0 ? QRCTM_ERR_CUDA : QRCTM_OK;
}

int qrctm_probe_fp64(int kind, int iters, double* tflops) {
  if (!tflops || iters < 1 || (kind != 0 && kind != 1)) return QRCTM_ERR_INVALID_ARG;
  int dev = 0, nsm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); return QRCTM_ERR_CUDA; }
  const int blocks = nsm * 2, threads = 256;
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
  CU(h, cudaMemsetAsync(h->flag, 0, 2 * sizeof(int), h->stream));
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
  int rc = ensure_s0(h); if (rc) return rc;
  rc = stage_eig_step(h, chi_new); if (rc) return rc;
  rc = check_flag(h); if (rc) return rc;
  CU(h, cudaMemsetAsync(h->s_prev, 0, sizeof(double) * h->chi_cap, h->stream));
  CU(h, cudaMemsetAsync(h->flag + 1, 0, sizeof(int), h->stream));       // a new convergence history starts here
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

int qrctm_chol_inv_f64(void* cuda_stream, int n, const double* G, double* R, double* Rinv, int* status, double* dev,
                       long long* prof) {
  if (!G || !R || !Rinv || !status || !dev || n < 1 || n > CHOL_MAX_N) return QRCTM_ERR_INVALID_ARG;
  if (chol_inv_attr() != cudaSuccess) { cudaGetLastError(); return QRCTM_ERR_CUDA; }
  chol_inv_kernel<<<1, CHOL_NT, chol_smem_bytes(n), static_cast<cudaStream_t>(cuda_stream)>>>(
      G, n, R, nullptr, Rinv, status, dev, nullptr, nullptr, 0.0, prof);
  return cudaGetLastError() == cudaSuccess ? QRCTM_OK : QRCTM_ERR_CUDA;
}

int qrctm_tridiag_f64(void* cuda_stream, int n, const double* C, double* d, double* e, long long* prof) {
  if (!C || !d || !e || n < 1 || n > TRI2_MAX_N) return QRCTM_ERR_INVALID_ARG;
  static bool attr = false;
  if (!attr) {
    if (cudaFuncSetAttribute(tridiag_smem2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)tri2_smem_bytes(TRI2_MAX_N)) != cudaSuccess) { cudaGetLastError(); return QRCTM_ERR_CUDA; }
    attr = true;
  }
  tridiag_smem2_kernel<<<1, TRI2_NT, tri2_smem_bytes(n), static_cast<cudaStream_t>(cuda_stream)>>>(C, n, d, e, prof);
  return cudaGetLastError() == cudaSuccess ? QRCTM_OK : QRCTM_ERR_CUDA;
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
  { int rc0 = ensure_s0(h); if (rc0) return rc0; }
  h->eig_rows = 0;
  const int chi = h->chi, b = h->b; const long long m = h->m, bc = (long long)b * chi;
  int m0, m1; shard_range(chi, rank, nranks, &m0, &m1);
  const int co = m1 - m0;
  // replicated: K1, K2 (0.3 % of the flops)
  int rc = stage_reduced_corner(h, h->C, h->T, h->X); if (rc) return rc;
  cudaError_t e;
  int rcq = stage_qr(h); if (rcq) return rcq;
  // the other ranks' rows of T' and the partial C' start from zero, so that either an all-gather of the slices or a
  // plain sum over ranks assembles the full tensors
  CU(h, cudaMemsetAsync(h->Tn, 0, sizeof(double) * m * chi, h->stream));
  CU(h, cudaMemsetAsync(h->Cn, 0, sizeof(double) * chi * chi, h->stream));
  if (co == 0) return QRCTM_OK;
  // this rank's slice: K3, K4, K5 with the columns [m0, m1) of Q in place of Q on the open leg.  An odd slice width is
  // padded with one zero column (cop): rows of 16-byte-aligned length keep every GEMM on the bulk-copy kernel.
  const int cop = (co & 1) && co < chi ? co + 1 : co;         // co == chi (one rank, odd chi): no room, no padding
  slice_cols_kernel<<<296, 256, 0, h->stream>>>(h->Q, m, chi, m0, co, cop, h->E);
  transpose_rows_kernel<<<(chi * cop + 255) / 256, 256, 0, h->stream>>>(h->R, chi, m0, co, cop, h->Rt);
  h->launches += 2;
  CU(h, cudaGetLastError());
  rc = stage_half_absorb(h, h->E, h->T, h->P, cop); if (rc) return rc;
  rc = stage_absorb_a(h, h->P, h->S, 0, nullptr, cop); if (rc) return rc;
  double* Tn_slice = h->Tn + (long long)m0 * bc;                       // rows (m, r), m in [m0, m1)
  rc = stage_project(h, h->S, h->Q, Tn_slice, cop, chi, co); if (rc) return rc;
  // partial (E4): W[(mo,r),n] = sum_k R[m0+mo,k] Q[k,(r,n)];  C'_part[p,n] = sum_{(mo,r)} T'[(mo,r),p] W[(mo,r),n]
  GemmCall c1{h->Q, bc, 1, h->Rt, cop, h->W, IndexMap{1, 1, 0}, plain_map(bc), (int)bc, cop, chi, 0};
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
