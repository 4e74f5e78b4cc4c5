// Host side of the NEXT-2 top-k symmetric eigensolver: workspace layout and the launch sequence (kernels: eigh.cuh).
// Part of the single translation unit qrctm_api.cu; included inside its anonymous namespace after qr_driver.cuh.
#pragma once

// ------------------------------------------------------------------ NEXT-2: top-k symmetric eigensolver
constexpr int EIGH_MAX_N = 14000;     // d, e2 of the multisection / two columns of the back-transform in shared memory
constexpr int EIGH_MAX_GROUPS = 96;   // row groups of the tridiagonalisation sweep (column partials of y per group)

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

// Launch with programmatic stream serialisation: the grid may be set up while its predecessor in the stream is still
// draining; the three tridiagonalisation kernels start with griddepcontrol.wait, which holds them until the
// predecessor has completed and its writes are visible (eigh.cuh, eigh_pdl_sync).
template <class... KArgs, class... Args>
void launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

// Householder tridiagonalisation of W (n x n symmetric, row-major, DEVICE; upper triangle swept, destroyed): diagonal
// -> wk.d, off-diagonal -> wk.e (e[i] couples i-1 and i), reflectors left in W / wk.tau.  Also K8's path for corner
// matrices too large for one SM's shared memory.  Returns kernels launched.
long long eigh_tridiagonalise(cudaStream_t st, int n, double* W, const EighWork& wk) {
  long long launches = 0;
  cudaMemsetAsync(wk.tau, 0, sizeof(double) * n, st);
#define REFL(k_, vprev_, vnew_)                                                                                  \
  do {                                                                                                           \
    const int left_ = n - (k_);                                                                                  \
    if (left_ <= 2048) launch_pdl(eigh_reflector_kernel<2>, dim3(1), dim3(1024), 0, st, W, n, (k_), wk.y, wk.rowpart, wk.colpart, rg_prev, (vprev_), wk.w, (vnew_), wk.tau, wk.d, wk.e); \
    else if (left_ <= 6144) launch_pdl(eigh_reflector_kernel<6>, dim3(1), dim3(1024), 0, st, W, n, (k_), wk.y, wk.rowpart, wk.colpart, rg_prev, (vprev_), wk.w, (vnew_), wk.tau, wk.d, wk.e); \
    else if (left_ <= 10240) launch_pdl(eigh_reflector_kernel<10>, dim3(1), dim3(1024), 0, st, W, n, (k_), wk.y, wk.rowpart, wk.colpart, rg_prev, (vprev_), wk.w, (vnew_), wk.tau, wk.d, wk.e); \
    else launch_pdl(eigh_reflector_kernel<14>, dim3(1), dim3(1024), 0, st, W, n, (k_), wk.y, wk.rowpart, wk.colpart, rg_prev, (vprev_), wk.w, (vnew_), wk.tau, wk.d, wk.e); \
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
    launch_pdl(eigh_pass_kernel, dim3(nch, ng), dim3(256), 0, st, W, n, k2, rg, vprev, wk.w, vnew, wk.rowpart, wk.colpart);
    if (nt <= 2048) { rg_prev = rg; launches += 2; }       // launch-latency-bound tail: one kernel fewer per step
    else {
      launch_pdl(eigh_ysum_kernel, dim3((nt + 63) / 64), dim3(64), 0, st, wk.rowpart, wk.colpart, n, k2, rg, wk.y);
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
  return launches;
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
  launches += eigh_tridiagonalise(st, n, W, wk);
  const int nc = 2 * k < n ? 2 * k : n;            // candidates: the k smallest and the k largest eigenvalues
  multisect_kernel<<<(nc + 3) / 4, 128, sizeof(double) * (2 * (size_t)n + 40), st>>>(wk.d, wk.e, n, wk.eig, k);
  eigh_select_kernel<<<(nc + 255) / 256, 256, 0, st>>>(wk.eig, nc, k, lam, wk.d, wk.e, n, wk.scal);
  eigh_invit_kernel<<<(k + 31) / 32, 32, 0, st>>>(wk.d, wk.e, n, lam, k, wk.scal, wk.Z, wk.U0, wk.U1, wk.U2, 3);
  launches += 4;
  *err = cudaGetLastError();
  if (*err != cudaSuccess) return -1;
  long long nq = qr_factor_blocked(st, 3, n, k, wk.Z, U, wk.R, wk.qr, err);      // Householder: clusters of near-parallel vectors
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

