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
  constexpr long long cap = (long long)QR_REG_RPT_TALL * (QR_REG_NT / QR_NB_REG);
  if (rows <= cap * reg_panel_max_cluster())
    return qr_factor_blocked_t<QR_NB_REG, true>(st, rows, n, X, Q, R, work, err);
  return qr_factor_blocked_t<QR_NB, false>(st, rows, n, X, Q, R, work, err);
}

