// The stages of one QR-CTMRG iteration as launches on the handle's stream: K1 (E1), K3/K4/K5 (E3), K4 layered
// (NEXT-1), K6 / K6' (E4 / E5+E4'), K7, K8, the step itself (do_step) and its CUDA-graph capture / replay.
// Part of the single translation unit qrctm_api.cu; included inside its anonymous namespace after the drivers.
#pragma once


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

// K2 (E2): X = Q R, diag(R) >= 0.  Automatic path: CholeskyQR2, with the Householder path as its fallback -- decided
// on the device: by the host after a synchronisation when launching directly, by a conditional graph node when the
// step is being captured (no host round trip in the replayed step).
int stage_qr(qrctm* h) {
  cudaError_t e;
  long long nl;
  if (h->qr_path == 1) {
    nl = qr_factor_level2(h->stream, h->m, h->chi, h->X, h->Q, h->R, h->qrwork, &e);
  } else {
    QrFallback fb{1, nullptr, nullptr};
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (h->stream && cudaStreamIsCapturing(h->stream, &cs) == cudaSuccess && cs == cudaStreamCaptureStatusActive) {
      if (!h->cap_aux) return fail(h, QRCTM_ERR_CUDA, "no auxiliary capture stream");
      fb = QrFallback{2, h->cap_aux, nullptr};
    } else if (h->cap_aux) {
      fb = QrFallback{3, h->cap_aux, &h->g_qrfb};       // direct launches: prebuilt {condition; IF Householder} graph
    }
    if (h->branch && h->stream) { fb.br = h->branch; fb.e_fork = h->ev_fork; fb.e_join = h->ev_join; }
    nl = qr_factor_blocked(h->stream, h->qr_path, h->m, h->chi, h->X, h->Q, h->R, h->qrwork, &e, fb);
  }
  if (nl < 0) return fail(h, QRCTM_ERR_CUDA, "qr", e);
  h->launches += nl;
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
// absorb mode 2 (automatic): the layered contraction does 4 d D^6 flops per (J, m) pair against 2 D^8, but as two short-K
// GEMMs (K = D^2 and d D^2) that reach ~55 % of the DMMA rate at D = 7 and far less below (K = 25 at D = 5 is two
// k-tiles); measured on a B200 it wins from D = 6 up (K4 at D = 5, chi = 100: 0.48 against 0.29 ms; D = 6, chi = 100: 1.1
// against 1.8 ms; D = 7, chi = 196: 1.8 against 12.7 ms), so that is the rule, with a 2x flop margin on d
bool use_layered(const qrctm* h) {
  if (!layered_ok(h)) return false;
  if (h->absorb_mode == 1) return true;
  return h->absorb_mode == 2 && h->D >= 6 && 4 * h->d <= h->b;
}

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
  g1.epi = 2;
  g1.resb = 1;
  GEMM(h, g1);
  GemmCall g2{h->P1, M2, 1, h->B2, h->L.ld2, S, IndexMap{chi * D, (long long)D * m, D}, IndexMap{D, m, 1},
              (int)M2, b, d * b, 0};
  g2.epi = 2;
  g2.resb = 1;
  GEMM(h, g2);
  return QRCTM_OK;
}

// K5: out[(m,r),n] = sum_{(J,d)} S''[(J,d),(m,r)] Qm[(J,d),n]
// chi_out: range of the index m of S'' (rows of out / D^2); ncols: columns of Qm (default: chi_out).
// chi_rows (<= chi_out): only the rows m < chi_rows of out are computed (a zero-padded slice, NEXT-4).
int stage_project(qrctm* h, const double* S, const double* Qm, double* out, int chi_out = 0, int ncols = 0,
                  int chi_rows = 0) {
  const int chi = chi_out > 0 ? chi_out : h->chi; const long long m = (long long)chi * h->b, mi = h->m;
  const int nq = ncols > 0 ? ncols : chi;
  const long long mrows = chi_rows > 0 ? (long long)chi_rows * h->b : m;
  GemmCall c{S, m, 1, Qm, nq, out, plain_map(nq), IndexMap{1, 1, 0}, (int)mrows, nq, (int)mi, 0};
  c.epi = 1;
  GEMM(h, c);
  return QRCTM_OK;
}

// K6 (E4): W[m,(r,n)] = sum_k R[m,k] Q[k,(r,n)] ;  C'[p,n] = sum_{(m,r)} T'[(m,r),p] W[(m,r),n]
// first half: W = R.Q needs only K2's outputs, so it can run on another stream beside K3..K5 (no scratch: no K split)
int stage_corner_accel_w(qrctm* h, cudaStream_t st) {
  const int chi = h->chi; const long long bc = (long long)h->b * chi;
  // W^T[(r,n), m] = sum_k Q[k,(r,n)] R^T[k,m]  (long index as M, both operands K-major); writes W
  transpose_small_kernel<<<(chi * chi + 255) / 256, 256, 0, st>>>(h->R, chi, h->Rt);
  h->launches += 1;
  GemmCall c1{h->Q, bc, 1, h->Rt, chi, h->W, IndexMap{1, 1, 0}, plain_map(bc), (int)bc, chi, chi, 0};
  cudaError_t ge;
  const int nl = launch_gemm(st, h->gemm_path, c1, nullptr, 0, &ge);
  if (nl < 0) return fail(h, QRCTM_ERR_CUDA, "gemm launch", ge);
  h->launches += nl;
  return QRCTM_OK;
}
int stage_corner_accel_c(qrctm* h) {
  const int chi = h->chi; const long long m = h->m;
  GemmCall c2{h->Tn, chi, 1, h->W, chi, h->Cn, plain_map(chi), IndexMap{1, 1, 0}, chi, chi, (int)m, 0};
  GEMM(h, c2);
  return QRCTM_OK;
}
int stage_corner_accel(qrctm* h) {
  int rc = stage_corner_accel_w(h, h->stream); if (rc) return rc;
  return stage_corner_accel_c(h);
}

// K6' (E5)+(E4'): Z = half_absorb(X), C~ = Z.a, Y = C~ Q, C' = Q^T Y.  K4's epilogue writes C~ transposed,
// S~[(k,r),(J,d)] = C~[(J,d),(k,r)], i.e. as the K x M operand of Y = C~ Q, so that this m x m x chi product runs on
// the same bulk-tensor-copy kernel (and stream-K schedule) as K5.
int stage_corner_enlarged(qrctm* h) {
  const int chi = h->chi; const long long m = h->m;
  int rc = stage_half_absorb(h, h->X, h->T, h->P); if (rc) return rc;
  rc = stage_absorb_a(h, h->P, h->S, 1); if (rc) return rc;          // S = C~^T
  GemmCall c1{h->S, m, 1, h->Q, chi, h->W, plain_map(chi), IndexMap{1, 1, 0}, (int)m, chi, (int)m, 0};
  c1.epi = 1;
  GEMM(h, c1);
  GemmCall c2{h->Q, chi, 1, h->W, chi, h->Cn, plain_map(chi), IndexMap{1, 1, 0}, chi, chi, (int)m, 0};
  GEMM(h, c2);
  return QRCTM_OK;
}

// K7: C,T <- sym(Cn,Tn) / ||.||_F
int stage_normalize(qrctm* h, const double* Cn, const double* Tn, bool record = false) {
  const int chi = h->chi, b = h->b;
  long long nT = (long long)chi * b * chi;
  int nbC = (int)(((long long)chi * chi + 255) / 256); if (nbC > 148) nbC = 148;
  int nbT = (int)((nT + 255) / 256); if (nbT > kPartialBlocks) nbT = kPartialBlocks;
  if (!h->small_off && nT + (long long)chi * chi <= 4096) {       // tiny: one CTA does K7 in one launch
    small_k7_kernel<<<1, SMALL_NT1, 0, h->stream>>>(Cn, Tn, chi, b, h->symmetrize, h->C, h->T, h->scal, h->flag,
                                                   record ? h->hist : nullptr, h->flag + 1, h->R);
    h->launches += 1;
    CU(h, cudaGetLastError());
    return QRCTM_OK;
  }
  sym_partial_kernel<<<nbC + nbT, 256, 0, h->stream>>>(Cn, Tn, chi, b, h->symmetrize, h->C, h->T, h->partial,
                                                      nbC, nbT);
  int nb = (int)((nT + (long long)chi * chi + 255) / 256); if (nb > 592) nb = 592;
  scale_kernel<<<nb, 256, 0, h->stream>>>(h->C, h->T, chi, b, h->partial, nbC, nbT, h->scal, h->flag,
                                          record ? h->hist : nullptr, h->flag + 1, h->R);
  h->launches += 2;
  CU(h, cudaGetLastError());
  return QRCTM_OK;
}

// K8: spectrum of h->C into s_out (+ delta against s_prev, optional update)
// to_host: the finalising kernel also writes delta and K7's flag word into the mapped pinned words h_pinned[0] / h_flag
// (the overlapped run driver then needs no copies after K8); *wrote_host says whether the selected path did.
int stage_spectrum(qrctm* h, double* s_out, int update_prev, cudaStream_t st, bool to_host = false, bool* wrote_host = nullptr) {
  double* hd = to_host ? h->h_pinned : nullptr;
  int* hf = to_host ? h->h_flag : nullptr;
  if (wrote_host) *wrote_host = false;
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
  if (chi <= SPEC_FUSED_MAX_N && !h->k8_old && !h->small_off) {
    static bool attrf = false;
    if (!attrf) {
      CU(h, cudaFuncSetAttribute(spectrum_fused_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)spectrum_fused_smem_bytes(SPEC_FUSED_MAX_N)));
      attrf = true;
    }
    // one warp per eigenvalue: 8 warps do for chi <= 8 (a 1024-thread CTA costs more to launch, to synchronise and to retire)
    spectrum_fused_kernel<<<1, chi <= 8 ? 256 : TRI2_NT, spectrum_fused_smem_bytes(chi), st>>>(h->C, chi, h->eig, s_out, h->s_prev, h->delta,
                                                                           update_prev, h->hist, h->flag + 1, hd, hf, h->flag);
    if (wrote_host) *wrote_host = to_host;
    h->launches += 1;
  } else if (chi <= TRI2_MAX_N && !h->k8_old) {
    static bool attr2 = false;
    if (!attr2) {
      CU(h, cudaFuncSetAttribute(tridiag_smem2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)tri2_smem_bytes(TRI2_MAX_N)));
      attr2 = true;
    }
    if (chi <= TRIR_MAX_N) tridiag_reg_kernel<2, 4, 16><<<1, 256, 0, st>>>(h->C, chi, h->dvec, h->evec);
    else if (chi <= TRIR_MAX_N2) tridiag_reg_kernel<4, 4, 32><<<1, 512, 0, st>>>(h->C, chi, h->dvec, h->evec);
    else tridiag_smem2_kernel<<<1, TRI2_NT, tri2_smem_bytes(chi), st>>>(h->C, chi, h->dvec, h->evec, nullptr);
    multisect_kernel<<<(chi + 3) / 4, 128, sizeof(double) * (2 * chi + 40), st>>>(h->dvec, h->evec, chi, h->eig);
    spectrum_finalize_kernel<<<1, nt, sizeof(double) * (chi + 40), st>>>(h->eig, chi, s_out, h->s_prev, h->delta,
                                                                        update_prev, h->hist, h->flag + 1, hd, hf, h->flag);
    if (wrote_host) *wrote_host = to_host;
    h->launches += 3;
  } else if (tri_bytes <= (size_t)max_smem && chi <= 1024) {
    tridiag_smem_kernel<<<1, 1024, tri_bytes, st>>>(h->C, chi, h->dvec, h->evec);
    multisect_kernel<<<(chi + 3) / 4, 128, sizeof(double) * (2 * chi + 40), st>>>(h->dvec, h->evec, chi,
                                                                                         h->eig);
    spectrum_finalize_kernel<<<1, nt, sizeof(double) * (chi + 40), st>>>(h->eig, chi, s_out, h->s_prev,
                                                                                 h->delta, update_prev, h->hist, h->flag + 1);
    h->launches += 3;
  } else if (h->k8work && chi <= 1024) {
    // corner too large for one SM's shared memory: the eigen step's multi-CTA tridiagonalisation (eigh_driver.cuh)
    // on a scratch copy, then the same multisection / finalisation as the fast path
    static bool ms_attr = false;
    if (!ms_attr) {
      CU(h, cudaFuncSetAttribute(multisect_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));
      ms_attr = true;
    }
    EighWork wk;
    eigh_layout(chi, 1, static_cast<char*>(h->k8work), &wk);
    CU(h, cudaMemcpyAsync(h->Wc, h->C, sizeof(double) * chi * chi, cudaMemcpyDeviceToDevice, st));
    h->launches += eigh_tridiagonalise(st, chi, h->Wc, wk);
    multisect_kernel<<<(chi + 3) / 4, 128, sizeof(double) * (2 * chi + 40), st>>>(wk.d, wk.e, chi, h->eig);
    spectrum_finalize_kernel<<<1, nt, sizeof(double) * (chi + 40), st>>>(h->eig, chi, s_out, h->s_prev, h->delta,
                                                                        update_prev, h->hist, h->flag + 1);
    h->launches += 2;
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

// Tiny problems: K1..K6 in one CTA (small_step.cuh).  Only with the default modes and when no per-stage events are wanted.
bool small_ok(qrctm* h) {
  if (h->small_off || h->gemm_path != 0 || h->corner_mode != 0 || h->absorb_mode == 1 || h->qr_path != 0) return false;
  // one CTA walks the chi dependent Householder columns and everything else of the step; from chi ~ 10 the general path
  // (CholeskyQR2 cluster kernel, small DMMA GEMMs, K8 beside the next step) is faster: measured per step at
  // (D, chi) = (2, 16) 98 us against 87, (3, 10) 96 / 82, (2, 24) 108 / 108, but (3, 7) 57 / 74, (2, 8) 47 / 60
  if (!h->small_force && h->chi > 8) return false;
  if (h->small_smem == 0) {
    int dev = 0, optin = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    h->small_smem = -1;
    if (optin > 0 &&
        cudaFuncSetAttribute(small_front_kernel<SMALL_NT1>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin) == cudaSuccess &&
        cudaFuncSetAttribute(small_front_kernel<SMALL_NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin) == cudaSuccess)
      h->small_smem = optin;
    cudaGetLastError();
  }
  return h->small_smem > 0 && sizeof(double) * small_front_doubles(h->b, h->chi) <= (size_t)h->small_smem;
}

int stage_small_front(qrctm* h) {
  const size_t smem = sizeof(double) * small_front_doubles(h->b, h->chi);
  if (h->m <= 40)
    small_front_kernel<SMALL_NT1><<<1, SMALL_NT1, smem, h->stream>>>(h->C, h->T, h->a_mat, h->L.lda_a, h->b, h->chi, h->X, h->Q,
                                                                   h->R, h->Tn, h->Cn);
  else
    small_front_kernel<SMALL_NT><<<1, SMALL_NT, smem, h->stream>>>(h->C, h->T, h->a_mat, h->L.lda_a, h->b, h->chi, h->X, h->Q,
                                                                 h->R, h->Tn, h->Cn);
  h->launches += 1;
  CU(h, cudaGetLastError());
  return QRCTM_OK;
}

int do_step(qrctm* h, cudaEvent_t* ev /* QRCTM_NSTAGE+1 events or null */, bool with_k7 = true) {
  if (!ev && small_ok(h)) {
    nvtxRangePushA("K1_K6_small");
    int rcs = stage_small_front(h);
    nvtxRangePop();
    if (rcs || !with_k7) return rcs;
    return stage_normalize(h, h->Cn, h->Tn, true);
  }
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
    rc = stage_qr(h);
  }
  // fork: K6's first product beside K3..K5 (not when per-stage events are wanted: the stage times would overlap)
  const bool forked = !rc && !ev && h->branch && h->corner_mode == 0 && h->stream != nullptr;
  if (forked) {
    if (cudaEventRecord(h->ev_fork, h->stream) != cudaSuccess || cudaStreamWaitEvent(h->branch, h->ev_fork, 0) != cudaSuccess)
      rc = fail(h, QRCTM_ERR_CUDA, "fork", cudaGetLastError());
    if (!rc) rc = stage_corner_accel_w(h, h->branch);
    if (!rc && cudaEventRecord(h->ev_join, h->branch) != cudaSuccess) rc = fail(h, QRCTM_ERR_CUDA, "fork", cudaGetLastError());
  }
  if (!rc) { mark(2, "K3_half_absorb"); rc = stage_half_absorb(h, h->Q, h->T, h->P); }
  if (!rc) {
    mark(3, "K4_absorb_a");
    rc = use_layered(h) ? stage_absorb_layered(h, h->P, h->S) : stage_absorb_a(h, h->P, h->S, 0);
  }
  if (!rc) { mark(4, "K5_project"); rc = stage_project(h, h->S, h->Q, h->Tn); }
  if (!rc) {
    mark(5, "K6_corner");
    if (forked) {
      if (cudaStreamWaitEvent(h->stream, h->ev_join, 0) != cudaSuccess) rc = fail(h, QRCTM_ERR_CUDA, "join", cudaGetLastError());
      if (!rc) rc = stage_corner_accel_c(h);
    } else rc = h->corner_mode == 0 ? stage_corner_accel(h) : stage_corner_enlarged(h);
  }
  if (!rc && !with_k7) { nvtxRangePop(); return rc; }
  if (!rc) { mark(6, "K7_normalize"); rc = stage_normalize(h, h->Cn, h->Tn, true); }
  if (!rc) mark(7, nullptr); else nvtxRangePop();
  return rc;
}

void invalidate_graphs(qrctm* h) {
  if (h->g_qrfb) { cudaGraphExecDestroy(h->g_qrfb); h->g_qrfb = nullptr; }
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
    if (!capture_graph(h, [&] { return stage_normalize(h, h->Cn, h->Tn, true); }, &h->g_k7, &h->g_k7_n)) h->graph_failed = 1;
  }
  int rc;
  if (can && h->g_k7) {
    CU(h, cudaGraphLaunch(h->g_k7, h->stream));
    h->launches += h->g_k7_n;
    rc = QRCTM_OK;
  } else {
    if (ev) { nvtxRangePushA("K7_normalize"); cudaEventRecord(ev[6], h->stream); }
    rc = stage_normalize(h, h->Cn, h->Tn, true);
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

