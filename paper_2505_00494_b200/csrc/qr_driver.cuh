// Host side of K2: workspace layout and the three QR drivers (per-reflector, blocked compact-WY with the
// register-resident cluster panel kernel, whole-matrix register kernel) plus the one-shot form-Q (kernels: qr_f64.cuh).
// Part of the single translation unit qrctm_api.cu; included inside its anonymous namespace after gemm_launch.cuh.
#pragma once


constexpr int QR_NB = 16;        // shared-memory / global panel kernel (fallback for very tall panels)
constexpr int QR_NB_REG = 16;    // register-resident panel kernel (default)
constexpr int QR_REG_NT = 256, QR_REG_RPT = 40;                       // 640 rows per CTA
constexpr int QR_REG_RPT_TALL = 80;                                   // 1280 rows per CTA (column k re-broadcast for the update)
constexpr int QR_MAX_PARTS = 320;

struct QrWork {     // carved out of the caller's work buffer
  double *V, *Vc, *tau, *Tfac, *W1, *W2, *splitk, *part, *Vct, *Gq, *Xq;
  size_t splitk_elems;
  // CholeskyQR2 (cholqr.cuh): R1 (upper), R1^-1, L2 (lower), R2^-1, deviations, status words
  double *cR1, *cRi1, *cL2, *cRi2, *cdev;
  int* cstat;       // [0] pass-1 breakdown, [1] pass-2 breakdown, [2] verdict: 1 = discard, take the Householder path
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
  size_t oc1 = take((size_t)n * n), oc2 = take((size_t)n * n), oc3 = take((size_t)n * n), oc4 = take((size_t)n * n);
  size_t ocd = take(8), ocs = take(8);
  if (w) {
    w->cR1 = reinterpret_cast<double*>(base + oc1); w->cRi1 = reinterpret_cast<double*>(base + oc2);
    w->cL2 = reinterpret_cast<double*>(base + oc3); w->cRi2 = reinterpret_cast<double*>(base + oc4);
    w->cdev = reinterpret_cast<double*>(base + ocd); w->cstat = reinterpret_cast<int*>(base + ocs);
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

template <int RPT>
cudaError_t launch_panel_reg_tall(cudaStream_t st, int C, double* V, long long ld, long long m, int j0, int nbw, double* Vc,
                                  double* tau, double* Tp, long long rpc) {
  auto k2 = qr_panel_reg2_kernel<QR_NB_REG, QR_REG_NT, RPT, true, false>;
  static bool attr2 = false;
  if (!attr2) {
    cudaError_t e = cudaFuncSetAttribute(k2, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
    attr2 = true;
  }
  cudaLaunchConfig_t cfg2 = {};
  cfg2.gridDim = dim3(C); cfg2.blockDim = dim3(QR_REG_NT); cfg2.dynamicSmemBytes = 0; cfg2.stream = st;
  cudaLaunchAttribute at2[1];
  at2[0].id = cudaLaunchAttributeClusterDimension;
  at2[0].val.clusterDim.x = C; at2[0].val.clusterDim.y = 1; at2[0].val.clusterDim.z = 1;
  cfg2.attrs = at2; cfg2.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg2, k2, V, ld, m, j0, nbw, Vc, tau, Tp, rpc);
}

cudaError_t launch_panel_reg(cudaStream_t st, double* V, long long ld, long long m, int j0, int nbw, double* Vc,
                             double* tau, double* Tp) {
  constexpr int cap = QR_REG_RPT * (QR_REG_NT / QR_NB_REG);
  const long long prow = m - j0;
  const int maxc = reg_panel_max_cluster();
  int C = 1;
  while (C < maxc && (prow + C - 1) / C > cap) C *= 2;
  const long long rpc = (prow + C - 1) / C;
  if (rpc > cap) {
    // tall panel: more rows per thread (48 / 64 / 80), column k re-broadcast for the update
    if (maxc < 16) return cudaErrorInvalidValue;
    constexpr int nrg = QR_REG_NT / QR_NB_REG;
    if (rpc <= 48 * nrg) return launch_panel_reg_tall<48>(st, C, V, ld, m, j0, nbw, Vc, tau, Tp, rpc);
    if (rpc <= 64 * nrg) return launch_panel_reg_tall<64>(st, C, V, ld, m, j0, nbw, Vc, tau, Tp, rpc);
    if (rpc <= QR_REG_RPT_TALL * nrg) return launch_panel_reg_tall<QR_REG_RPT_TALL>(st, C, V, ld, m, j0, nbw, Vc, tau, Tp, rpc);
    return cudaErrorInvalidValue;
  }
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

constexpr int wy_fused_max_slabs16 = 7;     // 16-CTA clusters co-resident on a B200 (launch__cluster_max_active)
// One-launch version (wy_fused_cluster_kernel): clusters of 8 CTAs, one per 16-column slab.  Returns 0 if the
// shape does not fit it (rows per thread, shared memory), else 1 after launching.
template <int NB, int RPT>
int launch_wy_fused(cudaStream_t st, const double* Vp, long long ldv, double* Y, long long ldy, long long rows, int nc,
                    int nbw, const double* Tp, int transT, cudaError_t* err) {
  // clusters of 8 (15 of them fit the GPU at once); taller matrices: clusters of 16 (7 at once) while the slabs fit
  // one wave of them -- beyond that the three streaming kernels are faster
  static int max16 = -1;
  if (max16 < 0) {
    max16 = cudaFuncSetAttribute(wy_fused_cluster_kernel<NB, RPT>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) ==
                    cudaSuccess ? 1 : 0;
    cudaGetLastError();
  }
  const int nslab_ = (nc + NB - 1) / NB;
  int CS = 8;
  if ((rows + CS - 1) / CS > 32 * RPT) {
    if (!max16 || nslab_ > wy_fused_max_slabs16) return 0;
    CS = 16;
  }
  const int rows_cta = (int)((rows + CS - 1) / CS);
  if (rows_cta > 32 * RPT) return 0;
  const size_t smem = sizeof(double) * ((size_t)rows_cta * (NB + 2) + 8 * 256 + 16 * 256 + 256);
  static int max_smem = -1;
  if (max_smem < 0) {
    int dev = 0; cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  }
  if (smem > (size_t)max_smem) return 0;
  static bool attr = false;
  if (!attr) {
    *err = cudaFuncSetAttribute(wy_fused_cluster_kernel<NB, RPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (*err != cudaSuccess) return -1;
    attr = true;
  }
  const int nslab = (nc + NB - 1) / NB;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(nslab * CS); cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  *err = cudaLaunchKernelEx(&cfg, wy_fused_cluster_kernel<NB, RPT>, Vp, ldv, Y, ldy, rows, nc, nbw, Tp, transT, rows_cta);
  return *err == cudaSuccess ? 1 : -1;
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
    if (n2 > 0) {    // trailing update: A2 <- (I - Vp T^T Vp^T) A2
      const double* Vp = wk.Vc + (long long)j0 * n + j0;
      double* A2 = wk.V + (long long)j0 * n + j0 + nbw;
      // up to 8 x 32 x 20 = 5120 rows: one cluster launch; taller (cfg4): the three streaming kernels (a 40-rows-per-
      // thread instantiation spills and takes 60 us per panel against their 33, profiles/r1_qr_panel_phases.md)
      int nf = 0;
      if (NB == 16) {
        nf = launch_wy_fused<16, 20>(st, Vp, n, A2, n, rows - j0, n2, nbw, Tp, 1, err);
        if (nf < 0) return -1;
      }
      launches += nf > 0 ? nf : apply_block_reflector<NB>(st, Vp, n, A2, n, rows - j0, n2, nbw, Tp, 1, wk);
    }
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
  if (npan <= 16) {
    static bool pipe_attr = false;
    if (!pipe_attr) {
      *err = cudaFuncSetAttribute(wy_formq_trsm_pipe_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
      if (*err != cudaSuccess) return -1;
      pipe_attr = true;
    }
    wy_formq_trsm_pipe_kernel<NB><<<npan, NB * NB, sizeof(double) * (size_t)npan * NB * NB * 3, st>>>(wk.Gq, wk.Tfac, wk.Vc,
                                                                                                    n, n, wk.Xq);
  } else {
    wy_formq_trsm_kernel<NB><<<npan, NB * NB, sizeof(double) * (size_t)npan * NB * NB * 2, st>>>(wk.Gq, wk.Tfac, wk.Vc, n,
                                                                                               n, wk.Xq);
  }
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

// How the caller wants the "CholeskyQR2 not accurate enough -> Householder" decision taken (it is made on the device):
//   mode 0: never fall back (the verdict word is still written);
//   mode 1: the host reads the verdict (synchronises the stream) and launches the Householder path if needed;
//   mode 2: the stream is being captured: the Householder path goes into the body of a conditional IF node of the
//           capturing graph (captured on the stream `aux`), executed only when the verdict says so;
//   mode 3: direct launches without a host round trip: a small graph {set condition; IF node with the Householder
//           path as its body} is built once (captured on `aux`), kept in *cache by the caller, and launched on the
//           stream after the CholeskyQR2 kernels.
struct QrFallback {
  int mode; cudaStream_t aux; cudaGraphExec_t* cache;
  // optional second stream + two events: the independent pieces of CholeskyQR2 (the transposes beside the Gram /
  // Cholesky chain, R = R2 R1 beside Q = Q1 R2^-1) are forked onto it
  cudaStream_t br = nullptr; cudaEvent_t e_fork = nullptr, e_join = nullptr;
};

long long qr_factor_householder(cudaStream_t st, int qr_path, long long rows, int n, const double* X, double* Q,
                                double* R, void* work, cudaError_t* err);

// On the capturing stream s: enqueue the kernel that sets the condition from the verdict word and append an IF node
// after it; later work captured on s depends on that node.  Returns the (empty) body graph of the IF node.
cudaError_t cholqr_append_cond(cudaStream_t s, const int* verdict, cudaGraph_t* body) {
  cudaStreamCaptureStatus cs; cudaGraph_t g = nullptr; const cudaGraphNode_t* deps = nullptr; size_t nd = 0;
  unsigned long long id = 0;
  cudaError_t e = cudaStreamGetCaptureInfo(s, &cs, &id, &g, &deps, &nd);
  if (e != cudaSuccess) return e;
  if (cs != cudaStreamCaptureStatusActive || !g) return cudaErrorInvalidValue;
  cudaGraphConditionalHandle hnd;
  e = cudaGraphConditionalHandleCreate(&hnd, g, 0, cudaGraphCondAssignDefault);
  if (e != cudaSuccess) return e;
  cholqr_set_cond_kernel<<<1, 32, 0, s>>>(hnd, verdict);
  e = cudaStreamGetCaptureInfo(s, &cs, &id, &g, &deps, &nd);
  if (e != cudaSuccess) return e;
  cudaGraphNodeParams prm = {};
  prm.type = cudaGraphNodeTypeConditional;
  prm.conditional.handle = hnd; prm.conditional.type = cudaGraphCondTypeIf; prm.conditional.size = 1;
  cudaGraphNode_t cn;
  e = cudaGraphAddNode(&cn, g, deps, nd, &prm);
  if (e != cudaSuccess) return e;
  e = cudaStreamUpdateCaptureDependencies(s, &cn, 1, cudaStreamSetCaptureDependencies);
  if (e != cudaSuccess) return e;
  *body = prm.conditional.phGraph_out[0];
  return cudaSuccess;
}

// Capture the Householder path into `body` on the stream aux.
cudaError_t cholqr_capture_body(cudaStream_t aux, cudaGraph_t body, long long rows, int n, const double* X, double* Q,
                                double* R, void* work) {
  cudaError_t e = cudaStreamBeginCaptureToGraph(aux, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
  if (e != cudaSuccess) return e;
  cudaError_t eh = cudaSuccess;
  const long long nh = qr_factor_householder(aux, 0, rows, n, X, Q, R, work, &eh);
  cudaGraph_t tmp = nullptr;
  e = cudaStreamEndCapture(aux, &tmp);
  if (nh < 0) return eh != cudaSuccess ? eh : cudaErrorUnknown;
  return e;
}

constexpr int kCholqrMinN = 48;
constexpr int kCholqrMinNCluster = 12;    // with the one-launch cluster kernel CholeskyQR2 wins from ~12 columns
constexpr double kCholqrDevMax = 1e-4;     // ||Q1^T Q1 - I||_F above this: cond(c~)^2 eps is not small, discard

cudaError_t chol_inv_attr() {
  static bool attr = false;
  if (attr) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(chol_inv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)chol_smem_bytes(CHOL_MAX_N));
  if (e == cudaSuccess) attr = true;
  return e;
}

// CholeskyQR2 (cholqr.cuh).  Returns launches on the main path, -1 on error, -2 if the shape does not fit.
long long qr_factor_cholqr2(cudaStream_t st, long long rows, int n, const double* X, double* Q, double* R, void* work,
                            cudaError_t* err, QrFallback fb) {
  if (n > CHOL_MAX_N || rows < n) return -2;
  QrWork wk;
  qr_layout(rows, n, static_cast<char*>(work), &wk);
  *err = chol_inv_attr();
  if (*err != cudaSuccess) return -1;
  const size_t smem = chol_smem_bytes(n);
  long long launches = 0;
  int nl;
  // small c~: the whole CholeskyQR2 in one cluster launch (cholqr.cuh) when 16 row slabs fit shared memory
  bool clustered = false;
  if (n <= CHOLC_MAX_N && rows >= 32) {
    static int optin = 0, c16 = -1;
    if (c16 < 0) {
      int dev = 0; cudaGetDevice(&dev);
      cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
      c16 = (cudaFuncSetAttribute(cholqr2_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - 1024) == cudaSuccess &&
             cudaFuncSetAttribute(cholqr2_cluster_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) ? 1 : 0;
      cudaGetLastError();
    }
    int C = 16;
    while (C > 2 && (rows + C / 2 - 1) / (C / 2) <= 48) C /= 2;          // at least ~48 rows per CTA
    const int rpc = (int)((rows + C - 1) / C);
    const size_t csm = cholqr2_cluster_smem_bytes(n, rpc);
    if (c16 == 1 && csm + 1024 <= (size_t)optin) {
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3(C); cfg.blockDim = dim3(CHOL_NT); cfg.dynamicSmemBytes = csm; cfg.stream = st;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      *err = cudaLaunchKernelEx(&cfg, cholqr2_cluster_kernel, X, rows, n, Q, R, wk.cstat, wk.cdev, kCholqrDevMax, rpc,
                                static_cast<long long*>(nullptr));
      if (*err != cudaSuccess) return -1;
      launches += 1;
      clustered = true;
    }
  }
  const dim3 tg((unsigned)((rows + 31) / 32), (n + 31) / 32), tb(32, 8);
  const bool fork_ok = fb.br != nullptr && fb.e_fork != nullptr && fb.e_join != nullptr && st != nullptr;
  if (!clustered) {
  // pass 1
  if (fork_ok) {                                   // X^T for the first product, beside Gram matrix and factorisation
    if (cudaEventRecord(fb.e_fork, st) != cudaSuccess || cudaStreamWaitEvent(fb.br, fb.e_fork, 0) != cudaSuccess) { *err = cudaGetLastError(); return -1; }
    transpose_tall_kernel<<<tg, tb, 0, fb.br>>>(X, rows, n, wk.Vct);
    if (cudaEventRecord(fb.e_join, fb.br) != cudaSuccess) { *err = cudaGetLastError(); return -1; }
  }
  nl = launch_gemm(st, 0, GemmCall{X, n, 1, X, n, wk.Gq, plain_map(n), IndexMap{1, 1, 0}, n, n, (int)rows, 0},
                   wk.splitk, wk.splitk_elems, err);
  if (nl < 0) return -1;
  launches += nl;
  chol_inv_kernel<<<1, CHOL_NT, smem, st>>>(wk.Gq, n, wk.cR1, nullptr, wk.cRi1, wk.cstat, wk.cdev, nullptr, nullptr, 0.0, nullptr);
  if (!fork_ok) transpose_tall_kernel<<<tg, tb, 0, st>>>(X, rows, n, wk.Vct);
  else if (cudaStreamWaitEvent(st, fb.e_join, 0) != cudaSuccess) { *err = cudaGetLastError(); return -1; }
  launches += 2;
  nl = launch_gemm(st, 0, GemmCall{wk.Vct, rows, 1, wk.cRi1, n, wk.V, plain_map(n), IndexMap{1, 1, 0}, (int)rows, n, n, 0},
                   wk.splitk, wk.splitk_elems, err);                                   // Q1 = X R1^-1
  if (nl < 0) return -1;
  launches += nl;
  // pass 2
  if (fork_ok) {                                   // Q1^T for the second product, beside Gram matrix and factorisation
    if (cudaEventRecord(fb.e_fork, st) != cudaSuccess || cudaStreamWaitEvent(fb.br, fb.e_fork, 0) != cudaSuccess) { *err = cudaGetLastError(); return -1; }
    transpose_tall_kernel<<<tg, tb, 0, fb.br>>>(wk.V, rows, n, wk.Vct);
    if (cudaEventRecord(fb.e_join, fb.br) != cudaSuccess) { *err = cudaGetLastError(); return -1; }
  }
  nl = launch_gemm(st, 0, GemmCall{wk.V, n, 1, wk.V, n, wk.Gq, plain_map(n), IndexMap{1, 1, 0}, n, n, (int)rows, 0},
                   wk.splitk, wk.splitk_elems, err);
  if (nl < 0) return -1;
  launches += nl;
  chol_inv_kernel<<<1, CHOL_NT, smem, st>>>(wk.Gq, n, nullptr, wk.cL2, wk.cRi2, wk.cstat + 1, wk.cdev + 1, wk.cstat,
                                            wk.cstat + 2, kCholqrDevMax, nullptr, kCholFastDsum);
  if (!fork_ok) transpose_tall_kernel<<<tg, tb, 0, st>>>(wk.V, rows, n, wk.Vct);
  else {
    if (cudaStreamWaitEvent(st, fb.e_join, 0) != cudaSuccess) { *err = cudaGetLastError(); return -1; }
    // R = R2 R1 = L2^T R1 beside Q = Q1 R2^-1 (no scratch: no K split on the side stream)
    if (cudaEventRecord(fb.e_fork, st) != cudaSuccess || cudaStreamWaitEvent(fb.br, fb.e_fork, 0) != cudaSuccess) { *err = cudaGetLastError(); return -1; }
    nl = launch_gemm(fb.br, 0, GemmCall{wk.cL2, n, 1, wk.cR1, n, R, plain_map(n), IndexMap{1, 1, 0}, n, n, n, 0}, nullptr, 0, err);
    if (nl < 0) return -1;
    launches += nl;
    if (cudaEventRecord(fb.e_join, fb.br) != cudaSuccess) { *err = cudaGetLastError(); return -1; }
  }
  launches += 2;
  nl = launch_gemm(st, 0, GemmCall{wk.Vct, rows, 1, wk.cRi2, n, Q, plain_map(n), IndexMap{1, 1, 0}, (int)rows, n, n, 0},
                   wk.splitk, wk.splitk_elems, err);                                   // Q = Q1 R2^-1
  if (nl < 0) return -1;
  launches += nl;
  if (!fork_ok) {
    nl = launch_gemm(st, 0, GemmCall{wk.cL2, n, 1, wk.cR1, n, R, plain_map(n), IndexMap{1, 1, 0}, n, n, n, 0},
                     wk.splitk, wk.splitk_elems, err);                                 // R = R2 R1 = L2^T R1
    if (nl < 0) return -1;
    launches += nl;
  } else if (cudaStreamWaitEvent(st, fb.e_join, 0) != cudaSuccess) { *err = cudaGetLastError(); return -1; }
  }
  *err = cudaGetLastError();
  if (*err != cudaSuccess) return -1;
  if (fb.mode == 1) {
    int verdict = 0;
    *err = cudaMemcpyAsync(&verdict, wk.cstat + 2, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (*err == cudaSuccess) *err = cudaStreamSynchronize(st);
    if (*err != cudaSuccess) return -1;
    if (verdict) {
      long long nh = qr_factor_householder(st, 0, rows, n, X, Q, R, work, err);
      if (nh < 0) return -1;
      launches += nh;
    }
  } else if (fb.mode == 2) {
    cudaGraph_t body = nullptr;
    *err = cholqr_append_cond(st, wk.cstat + 2, &body);
    if (*err != cudaSuccess) return -1;
    launches += 1;
    *err = cholqr_capture_body(fb.aux, body, rows, n, X, Q, R, work);
    if (*err != cudaSuccess) return -1;
  } else if (fb.mode == 3) {
    if (!*fb.cache) {
      cudaGraph_t g = nullptr, body = nullptr, tmp = nullptr;
      *err = cudaGraphCreate(&g, 0);
      if (*err != cudaSuccess) return -1;
      *err = cudaStreamBeginCaptureToGraph(fb.aux, g, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
      if (*err == cudaSuccess) {
        const cudaError_t e1 = cholqr_append_cond(fb.aux, wk.cstat + 2, &body);
        const cudaError_t e2 = cudaStreamEndCapture(fb.aux, &tmp);
        *err = e1 != cudaSuccess ? e1 : e2;
      }
      if (*err == cudaSuccess) *err = cholqr_capture_body(fb.aux, body, rows, n, X, Q, R, work);
      if (*err == cudaSuccess) *err = cudaGraphInstantiate(fb.cache, g, 0);
      cudaGraphDestroy(g);
      if (*err != cudaSuccess) { *fb.cache = nullptr; return -1; }
    }
    *err = cudaGraphLaunch(*fb.cache, st);
    if (*err != cudaSuccess) return -1;
    launches += 1;
  }
  return launches;
}

// qr_path: 0 = automatic (CholeskyQR2 when c~ has kCholqrMinN..CHOL_MAX_N columns, Householder when that is discarded
// or does not fit), 2 = Householder blocked path only, 3 = Householder automatic (whole-matrix register kernel when it
// fits, else blocked) -- the round-1 default, 4 = CholeskyQR2 whenever it fits (any n <= CHOL_MAX_N)
long long qr_factor_blocked(cudaStream_t st, int qr_path, long long rows, int n, const double* X, double* Q,
                            double* R, void* work, cudaError_t* err, QrFallback fb = QrFallback{1, nullptr, nullptr}) {
  // below ~48 columns the whole QR is launch-latency bound and the single-launch register-resident Householder
  // kernel wins (cfg0: 44 us against 71 us, cfg1: 119 against 133; measured, profiles/r2_k2_cholqr2.md)
  if (qr_path == 0 && (n >= kCholqrMinN || (n >= kCholqrMinNCluster && n <= CHOLC_MAX_N && rows >= 32 &&
                        cholqr2_cluster_smem_bytes(n, (int)((rows + 15) / 16)) + 2048 <= (size_t)227 * 1024))) {
    const long long nl = qr_factor_cholqr2(st, rows, n, X, Q, R, work, err, fb);
    if (nl != -2) return nl;
  }
  if (qr_path == 4) {
    const long long nl = qr_factor_cholqr2(st, rows, n, X, Q, R, work, err, fb);
    if (nl != -2) return nl;
  }
  return qr_factor_householder(st, qr_path == 3 ? 0 : qr_path, rows, n, X, Q, R, work, err);
}

// Householder paths.  qr_path: 0 = whole-matrix register kernel when it fits, else blocked; 2 = always blocked
long long qr_factor_householder(cudaStream_t st, int qr_path, long long rows, int n, const double* X, double* Q,
                                double* R, void* work, cudaError_t* err) {
  if (qr_path == 0 && n <= 112) {
    QrWork wk;
    qr_layout(rows, n, static_cast<char*>(work), &wk);
    long long nl = n <= 32 ? qr_factor_fullreg_t<2, 24>(st, rows, n, X, Q, R, wk, err)
                 : n <= 64 ? qr_factor_fullreg_t<4, 16>(st, rows, n, X, Q, R, wk, err)
                           : qr_factor_fullreg_t<7, 10>(st, rows, n, X, Q, R, wk, err);
    if (nl != -2) return nl;
  }
  constexpr long long cap = (long long)QR_REG_RPT_TALL * (QR_REG_NT / QR_NB_REG);
  if (rows <= cap * reg_panel_max_cluster())
    return qr_factor_blocked_t<QR_NB_REG, true>(st, rows, n, X, Q, R, work, err);
  return qr_factor_blocked_t<QR_NB, false>(st, rows, n, X, Q, R, work, err);
}

