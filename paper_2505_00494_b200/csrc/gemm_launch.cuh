// Host side of the FP64 GEMM: tile-configuration choice, split-K cost model, launches (kernels: gemm_f64.cuh).
// Part of the single translation unit qrctm_api.cu; included inside its anonymous namespace.
#pragma once

// ------------------------------------------------------------------ GEMM launcher

// Launch with programmatic stream serialisation (kernels: pdl_sync() in gemm_f64.cuh).
template <class... KArgs, class... Args>
cudaError_t pdl_launch(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

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
  return pdl_launch(gemm_f64_dmma<BM, BN, WM, WN, STAGES>, grid, dim3(NT), smem, st, g);
}

// Tensor maps for the tiled bulk copies of the ws kernel (the encoder comes from the driver through the runtime, the
// library links no libcuda).  Returns false if the driver entry point is missing or the shape is refused.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
bool encode_operand_map(CUtensorMap* tm, const double* base, long long ld, int width, int krows, int box_w) {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(f);
    cudaGetLastError();
  }
  if (!fn || width < 1 || krows < 1) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)width, (cuuint64_t)krows};
  const cuuint64_t strides[1] = {(cuuint64_t)ld * sizeof(double)};
  const cuuint32_t box[2] = {(cuuint32_t)box_w, (cuuint32_t)BK};
  const cuuint32_t estr[2] = {1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// stream-K request: workspace for the partial tiles; `used` is set when the launch went that way (else plain tiles)
struct StreamK { double* ws; size_t ws_elems; bool used; bool hybrid; };

template <int BM, int BN, int WM, int WN, int STAGES>
cudaError_t launch_cfg_ws(cudaStream_t st, const GemmArgs& g, int splits, StreamK* sk = nullptr) {
  constexpr int NT = ((BM / WM) * (BN / WN) + 1) * 32;
  constexpr size_t smem = sizeof(double) * STAGES * BK * ((BM + PAD) + (BN + PAD)) + (2 * STAGES + 2) * sizeof(uint64_t) +
                          sizeof(double) * (BM / WM) * (BN / WN) * 8 * (WN + 4) +     // + per-warp epilogue slabs
                          sizeof(long long) * (BM + BN);                               // + output-offset table
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
  // tiled bulk tensor copies when the k-rows are the stored rows (no K-row map, no batch offsets)
  ga.tma = 0;
  if (!g.batch && g.ka.div == 1 && g.ka.hi == 1 && g.ka.lo == 0)
    ga.tma = encode_operand_map(&ga.tmA, g.A, g.lda, g.M, g.K, BM + PAD) &&
             encode_operand_map(&ga.tmB, g.B, g.ldb, g.N, g.K, BN + PAD) ? 1 : 0;
  const long long nwork = (long long)((g.N + BN - 1) / BN) * ((g.M + BM - 1) / BM) * splits;
  if (sk) {
    // stream-K: one CTA per slot, every CTA the same number (+-1) of k-tiles; then the fix-up of the split tiles
    const int tn = (g.N + BN - 1) / BN, nkt = (g.K + BK - 1) / BK;
    const long long units = nwork * nkt;
    // hybrid: whole waves of tiles as they are, only the ragged last wave dealt out by k-tiles
    const long long t1 = sk->hybrid ? nwork / nslots * nslots : 0;
    const long long nsk = units - t1 * nkt < nslots ? units - t1 * nkt : nslots;      // stream-K CTAs
    const long long ncta = t1 + nsk;
    sk->used = splits == 1 && !g.batch && nsk >= 1 && nsk <= SK_MAXSEG && (size_t)2 * nsk * BM * BN <= sk->ws_elems;
    if (sk->used) {
      static bool sk_attr = false;
      if (!sk_attr) {
        cudaError_t e = cudaFuncSetAttribute(gemm_f64_dmma_ws<BM, BN, WM, WN, STAGES, true>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        sk_attr = true;
      }
      ga.sk = 1; ga.sk_ws = sk->ws; ga.sk_t1 = (int)t1;
      cudaError_t e1 = pdl_launch(gemm_f64_dmma_ws<BM, BN, WM, WN, STAGES, true>, dim3((unsigned)ncta), dim3(NT), smem, st, ga);
      if (e1 != cudaSuccess) return e1;
      return pdl_launch(streamk_fixup, dim3((unsigned)(nwork - t1), 8), dim3(256), 0, st, (const double*)sk->ws, BM, BN, tn, nkt,
                        units, (int)ncta, (int)t1, g.M, g.N, g.out, g.ro, g.co, g.mode);
    }
  }
  (void)nslots;                                  // one work item per CTA: the hardware scheduler balances better
  const unsigned grid = (unsigned)nwork;         // than a static persistent loop, with or without a start-up stagger
                                                 // between the two CTAs of an SM (measured, profiles/r1_gemm_experiments.md)
  return pdl_launch(gemm_f64_dmma_ws<BM, BN, WM, WN, STAGES>, dim3(grid), dim3(NT), smem, st, ga);
}

// Resident-B persistent launch (kernel: RESB = true): N <= BN, K short enough for all of B to sit in shared memory.
// Returns cudaErrorInvalidValue when the shape does not qualify (the caller then takes the ordinary launch).
template <int BM, int BN, int WM, int WN, int STAGES>
cudaError_t launch_cfg_ws_resb(cudaStream_t st, const GemmArgs& g, int nz) {
  constexpr int NT = ((BM / WM) * (BN / WN) + 1) * 32;
  const int nkt = (g.K + BK - 1) / BK;
  if (g.N > BN || nkt > 8) return cudaErrorInvalidValue;
  const size_t smem = sizeof(double) * BK * (STAGES * (BM + PAD) + (size_t)nkt * (BN + PAD)) + (2 * STAGES + 2) * sizeof(uint64_t) +
                      sizeof(double) * (BM / WM) * (BN / WN) * 8 * (WN + 4) + sizeof(long long) * (BM + BN);
  auto kern = gemm_f64_dmma_ws<BM, BN, WM, WN, STAGES, false, true>;
  static bool attr_done = false;
  static size_t max_smem = 0;
  if (!attr_done) {
    int dev = 0, optin = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    if (e != cudaSuccess) return e;
    max_smem = (size_t)optin;
    attr_done = true;
  }
  if (smem > max_smem) return cudaErrorInvalidValue;
  static int nsm = 0;
  if (!nsm) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev); }
  int per = 1;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, kern, NT, smem);
  if (per < 1) return cudaErrorInvalidValue;
  GemmArgs ga = g;
  ga.nz = nz;
  ga.tma = 0;
  if (!g.batch && g.ka.div == 1 && g.ka.hi == 1 && g.ka.lo == 0)
    ga.tma = encode_operand_map(&ga.tmA, g.A, g.lda, g.M, g.K, BM + PAD) &&
             encode_operand_map(&ga.tmB, g.B, g.ldb, g.N, g.K, BN + PAD) ? 1 : 0;
  const long long nwork = (long long)((g.M + BM - 1) / BM) * nz;
  const long long slots = (long long)nsm * per;
  const unsigned grid = (unsigned)(nwork < slots ? nwork : slots);
  return pdl_launch(kern, dim3(grid), dim3(NT), smem, st, ga);
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
  int resb = 0;                        // 1: short K, N within one tile: prefer the resident-B persistent kernel
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
  if (c.epi == 2) {
    // dense-block epilogue: columns in groups of wc with unit stride inside a group, rows with stride wc inside a row
    // group; every piece a bulk store may start at or cover must be 16-byte aligned: even strides, even M, even row groups
    const bool c3 = c.co.div0 > 1;
    const int wc = c3 ? c.co.div0 : c.co.div;
    const long long cin = c3 ? c.co.lo0 : c.co.lo, rin = c.ro.div0 > 1 ? -1 : c.ro.lo;
    const bool ok = c.mode == 0 && wc >= 1 && wc < 128 && c.N % wc == 0 && cin == 1 && rin == wc && c.M % 2 == 0 &&
                    c.ro.div % 2 == 0 && c.ro.hi % 2 == 0 && c.co.hi % 2 == 0 && (!c3 || c.co.lo % 2 == 0) && c.zo % 2 == 0 &&
                    (reinterpret_cast<uintptr_t>(c.out) & 15) == 0;
    if (ok) { g.dense_wc = wc; g.dense_magic = (65536 + wc - 1) / wc; }
    else g.epi = 1;
  }
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
  bool use_sk = false, sk_hybrid = false;
  int cfg = 0;          // 0: 64x64 cp.async, 1: 128x128 cp.async, 2: ws 128x128, 3: ws 128x104, 4: ws 128x64 (2 CTA/SM),
                        // 5: ws 128x56, 6: ws 80x208 (one wave for M <= 148 x 80, N <= 208), 7: ws 64x160
  const bool ws_big = ws_ok && c.M >= 96 && c.N >= 32 && (double)c.M * c.N * c.K > 2.0e8;
  if (c.batch > 0) {
    // batched launch (layered absorption): bulk-copy kernel only, one batch per gridDim.z, no split-K
    if (!ws_ok) { *err = cudaErrorInvalidValue; return -1; }
    const int pad128 = (c.N + 127) / 128 * 128, pad104 = (c.N + 103) / 104 * 104, pad64 = (c.N + 63) / 64 * 64;
    if (c.resb && c.N > 64 && c.N <= 104) {
      *err = launch_cfg_ws_resb<64, 104, 16, 104, 3>(st, g, c.batch);
      if (*err == cudaSuccess) return 1;
      if (*err != cudaErrorInvalidValue) return -1;
      cudaGetLastError();
    }
    if (c.N <= 56) *err = launch_cfg_ws<128, 56, 32, 56, 3>(st, g, c.batch);
    else if (pad64 <= pad104 && pad64 <= pad128) *err = launch_cfg_ws<128, 64, 64, 32, 4>(st, g, c.batch);
    else if (pad104 <= pad128 && nkt <= 6) *err = launch_cfg_ws<64, 104, 16, 104, 3>(st, g, c.batch);   // 2 CTAs/SM
    else if (pad104 <= pad128) *err = launch_cfg_ws<128, 104, 16, 104, 4>(st, g, c.batch);
    else *err = launch_cfg_ws<128, 128, 64, 32, 4>(st, g, c.batch);
    return *err == cudaSuccess ? 1 : -1;
  }
  if (ws_big && c.resb && c.N <= 56) {
    *err = launch_cfg_ws_resb<128, 56, 32, 56, 2>(st, g, 1);
    if (*err == cudaSuccess) return 1;
    if (*err != cudaErrorInvalidValue) return -1;
    cudaGetLastError();
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
    // 128 < N <= 160 (K5, chi = 150: 208 or 256 padded columns otherwise): 64 x 160 tiles, eight warps of 32 x 40
    // (a 128 x 160 tile needs 160 accumulator registers per thread with eight warps -- a 288-thread CTA gets 168 -- and
    // spills with sixteen warps at 96)
    if ((cfg == 2 || cfg == 3) && c.N > 128 && padded(160) * 100 < padded(bn) * 90) { bn = 160; cfg = 7; }
    const int bm = cfg == 7 ? 64 : 128;
    const long long tiles = (long long)((c.M + bm - 1) / bm) * ((c.N + bn - 1) / bn);
    const int slots = (cfg == 4 || cfg == 5) ? 296 : 148;
    const double t_kt = 2.1e-6 * bn / 128.0 * bm / 128.0 * ((cfg == 4 || cfg == 5) ? 2.0 : 1.0), t_fix = 4e-6;
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
    // stream-K instead when the tiles fill only a few ragged waves: every CTA gets the same share of k-tiles
    const double units = (double)tiles * nkt;
    if (tiles < 6LL * slots && units >= 24.0 * slots && (size_t)2 * slots * 128 * bn <= splitk_elems) {
      // up to two partial tiles per CTA written and read again, one more launch
      const double t_sk = ceil(units / slots) * t_kt + 2 * t_fix + 2.0 * (2.0 * slots * 128.0 * bn * 8.0) / 3e12 + 5e-6;
      if (t_sk < best * 0.97) { use_sk = true; splits = 1; }
    } else if (splits == 1 && tiles > slots && (size_t)2 * slots * 128 * bn <= splitk_elems) {
      // many waves: if the last one is ragged and long enough to be worth splitting, deal it out by k-tiles
      const long long rem = tiles % slots;
      if (rem > 0 && rem * 10 < slots * 8 && (double)rem * nkt >= 24.0 * slots) { use_sk = true; sk_hybrid = true; }
    }
    // N in (104, 208] with just over one wave of 128 x 104 tiles and no K split (K1, K6's first product, the form-Q
    // GEMM: 152 tiles on 148 SMs = two waves): 80 x 208 tiles cover N in one tile and M in one wave
    if (cfg == 3 && splits == 1 && !use_sk && c.N > 104 && c.N <= 208 && tiles > slots && tiles <= 2 * slots &&
        (c.M + 79) / 80 <= slots) {
      cfg = 6;
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
  StreamK skreq{splitk_ws, splitk_elems, false, sk_hybrid};
  StreamK* sk = use_sk ? &skreq : nullptr;
  switch (cfg) {
    case 2: *err = launch_cfg_ws<128, 128, 64, 32, 4>(st, g, splits, sk); break;
    case 3: *err = launch_cfg_ws<128, 104, 16, 104, 4>(st, g, splits, sk); break;
    case 4: *err = launch_cfg_ws<128, 64, 64, 32, 4>(st, g, splits, sk); break;
    case 5: *err = launch_cfg_ws<128, 56, 32, 56, 3>(st, g, splits, sk); break;
    case 6: *err = launch_cfg_ws<80, 208, 16, 104, 3>(st, g, splits, sk); break;
    case 7: *err = launch_cfg_ws<64, 160, 32, 40, 4>(st, g, splits, sk); break;
    case 1: *err = launch_cfg<128, 128, 64, 32, 4>(st, g, splits); break;
    default: *err = launch_cfg<64, 64, 32, 16, 4>(st, g, splits); break;
  }
  if (*err != cudaSuccess) return -1;
  ++launched;
  if (skreq.used) ++launched;
  if (splits > 1) {
    long long n = (long long)c.M * c.N;
    *err = pdl_launch(reduce_splitk, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, st, (const double*)splitk_ws, g.split_stride,
                      splits, c.M, c.N, c.out, c.ro, c.co, c.mode);
    if (*err != cudaSuccess) return -1;
    ++launched;
  }
  return launched;
}

