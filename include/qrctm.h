/* qrctm.h -- C ABI of the B200-native QR-CTMRG library (libqrctm.so).
 *
 * One C4v-symmetric QR-CTMRG iteration for a single-site real iPEPS, FP64, one
 * GPU, as defined in "Accelerating two-dimensional tensor network contractions
 * using QR-decompositions" (arXiv 2505.00494; PAPER.md below is
 * /root/reference/PAPER.md).  Equation labels (E0)..(E5) are the index-form
 * statement of the paper's Fig. 1 given in DESIGN.md section 2.
 *
 * Notation: d physical dim, D bond dim, b = D*D, chi boundary dim, m = chi*b.
 * All arrays are C-order (row-major) FP64.
 *   A[d][D][D][D][D]   site tensor, aux legs cyclic (up,left,down,right)
 *   C[chi][chi]        corner (symmetric)
 *   T[chi][b][chi]     edge, T[i][s][k] = T[k][s][i]
 *   Q[chi*b][chi]      isometry of the last step (rows (j,u))
 *   R[chi][chi]        upper triangular, diag(R) >= 0
 *
 * Pointers.  Every `double*` argument may be a HOST pointer or a DEVICE pointer
 * (e.g. torch tensor .data_ptr()); the library finds out which with
 * cudaPointerGetAttributes and copies accordingly.  Nothing the caller passes
 * is retained after the call returns (set_* copy in, get_* copy out).  The
 * handle owns all device workspaces; they are allocated in qrctm_create (or
 * taken from the caller through qrctm_create_in) and nothing is allocated in
 * qrctm_step / qrctm_run.
 *
 * Errors.  Every function returns an int status: QRCTM_OK (0) or a negative
 * code.  qrctm_last_error gives a text for the last failure on that handle.
 * No exceptions, no abort, nothing is printed.  Not converging within
 * max_iter is NOT an error.
 *
 * Determinism.  Same inputs give bitwise-identical outputs run to run: all
 * reductions use fixed trees, there are no floating-point atomics.
 *
 * There is no CPU fallback: without a CUDA device qrctm_create fails with
 * QRCTM_ERR_CUDA.
 *
 * Limits of this build: D <= 32, chi <= 800, d <= 64.  ONE DEVICE PER PROCESS: the
 * one-time kernel attributes (shared-memory opt-in, cluster sizes, occupancy) are
 * cached per process, so all handles of a process must live on the same device
 * (the one current at the first call); qrctm_create on a different device returns
 * QRCTM_ERR_INVALID_ARG.
 */
#ifndef QRCTM_H
#define QRCTM_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qrctm qrctm_t; /* opaque */

enum {
  QRCTM_OK = 0,
  QRCTM_ERR_INVALID_ARG = -1, /* null pointer, d/D/chi < 1, size overflow, bad option      */
  QRCTM_ERR_NOT_READY = -2,   /* step/run before set_A and set_env                         */
  QRCTM_ERR_CUDA = -3,        /* a CUDA call failed; see qrctm_last_error                  */
  QRCTM_ERR_NUMERIC = -4      /* NaN/Inf or zero Frobenius norm of C' or T'                */
};

/* Options for qrctm_set_option. */
enum {
  QRCTM_OPT_CORNER_MODE = 1, /* 0 = accelerated (E4) [default], 1 = enlarged corner (E5)+(E4')          */
  QRCTM_OPT_SYMMETRIZE = 2,  /* 1 [default] = symmetrise C', T' before normalising, 0 = only normalise   */
  QRCTM_OPT_CHECK_EVERY = 3, /* qrctm_run computes the corner spectrum / delta every n steps, default 1 */
  QRCTM_OPT_GEMM_PATH = 4,   /* 0 = FP64 tensor-core (DMMA) tiles [default], 1 = plain DFMA reference kernel */
  QRCTM_OPT_TIME_STAGES = 5, /* 1 = qrctm_run records CUDA events around every stage of every step (default 0) */
  QRCTM_OPT_QR_PATH = 6,     /* 0 [default] = automatic: CholeskyQR2 (two Gram / Cholesky / triangular-inverse passes, the
                                O(m chi^2) work on the DMMA GEMM; for chi <= 64 and m chi small enough one cluster launch with the
                                rows resident in shared memory) when 48 <= chi <= 208 (12 <= chi with the cluster kernel), checked on the device
                                (||Q1^T Q1 - I||_F <= 1e-4 and no pivot breakdown) and replaced by the Householder path
                                when the check fails (ill-conditioned or rank-deficient c~); Householder (as 3) outside
                                that range; 1 = one kernel launch per Householder reflector (slow reference path for
                                cross-checking); 2 = blocked compact-WY Householder with the cluster panel kernel;
                                3 = Householder automatic (whole-matrix register-resident cluster kernel when c~ fits:
                                chi <= 112, rows <= 16 x 160..384, else 2); 4 = CholeskyQR2 for any chi <= 208 */
  QRCTM_OPT_OVERLAP_CHECK = 7, /* 1 [default] = qrctm_run overlaps the convergence check of step k (side stream) with
                                K1..K6 of step k+1; results are identical, Q/R/raw buffers then hold the factors of
                                the last *started* iteration.  0 = strictly serial */
  QRCTM_OPT_USE_GRAPH = 8,   /* 1 [default] = K1..K6 and K7 are captured once into CUDA graphs and replayed by
                                qrctm_step / qrctm_run (needs a non-default stream); 0 = plain launches, which keep
                                the per-stage NVTX ranges for profilers */
  QRCTM_OPT_K8_PATH = 10,    /* K8 tridiagonalisation for chi <= 216: 0 [default] = the round-2 kernels (chi <= 24 fused
                                into one launch, chi <= 128 register-resident kernels, else thread-per-column kernel with un-
                                normalised reflectors), 1 = the round-1 kernel (for cross-checks) */
  QRCTM_OPT_SMALL_PATH = 11, /* 0 [default] = problems with chi <= 8 whose whole working set fits one CTA's shared memory
                                (2 m^2 + D^8 + 5 m chi doubles <= ~200 KB; cfg0) run K1..K6 as ONE kernel and K7 as one
                                more (plain DFMA loops, Householder QR) when the default modes are selected;
                                1 = always the general multi-kernel path; 2 = the one-kernel path whenever the working
                                set fits (e.g. D = 2, chi <= 24), also where the general path was measured faster */
  QRCTM_OPT_ABSORB_MODE = 9  /* K4: 0 [default] = contract with the explicit double-layer tensor a (2 chi^2 D^8 flops),
                                1 = layered: contract with the ket and the bra copy of A in turn (4 d chi^2 D^6
                                flops; same T' up to rounding; needs even chi, otherwise mode 0 is used),
                                2 = automatic: layered where it was measured faster on a B200: D >= 6 (and 4 d <= D^2,
                                even chi), explicit otherwise */
};

/* Create a handle for dimensions (d, D, chi); allocates every workspace with
 * cudaMalloc on the current device (about 32*(chi*D*D)^2 bytes: the two m x m
 * intermediates P and S plus the 2 m^2 intermediate of the layered mode, plus
 * 16*D^8 for the double-layer tensors; qrctm_workspace_bytes gives the exact
 * figure).  *out = NULL on failure. */
int qrctm_create(int d, int D, int chi, qrctm_t** out);

/* Bytes of device workspace a handle for (d, D, chi) needs (for callers that
 * own the memory, e.g. a torch tensor).  Returns 0 on invalid arguments. */
unsigned long long qrctm_workspace_bytes(int d, int D, int chi);

/* Same as qrctm_create, but all device workspaces are carved out of the
 * caller's DEVICE buffer `workspace` (>= qrctm_workspace_bytes, 256-byte
 * aligned), which must outlive the handle.  This is how the Python binding
 * lets PyTorch own device memory. */
int qrctm_create_in(int d, int D, int chi, void* workspace,
                    unsigned long long workspace_bytes, qrctm_t** out);

int qrctm_destroy(qrctm_t* h);

/* All later work of this handle is enqueued on `cuda_stream` (a cudaStream_t,
 * e.g. torch.cuda.current_stream().cuda_stream).  Default: the legacy stream. */
int qrctm_set_stream(qrctm_t* h, void* cuda_stream);

/* K0.  Copy A in and build the double-layer tensor (E0)
 *   a[(u u')][(l l')][(d d')][(r r')] = sum_s A[s][u][l][d][r] A[s][u'][l'][d'][r']
 * (Fig. 1(b)).  Keeps the current environment C, T (the paper's
 * optimiser reuses it across updates of A). */
int qrctm_set_A(qrctm_t* h, const double* A);

/* Copy an initial environment in, symmetrise (if enabled) and Frobenius-
 * normalise it, reset the convergence history: the previous spectrum becomes the
 * spectrum of this C (computed by the next qrctm_run under its first step, or by
 * whichever other entry is the first to overwrite C).  delta is always measured
 * against the spectrum of the previous check, or of this C before the first one. */
int qrctm_set_env(qrctm_t* h, const double* C, const double* T);

/* One QR-CTMRG iteration, asynchronous on the stream:
 *   (E1) c~[(j,u),k] = sum_i C[j,i] T[i,u,k]
 *   (E2) c~ = Q R, unpivoted Householder QR, then signs fixed so diag(R) >= 0
 *   (E3) T'[m,r,n] = sum Q[(j,u),m] T[j,l,J] a[u,l,d,r] Q[(J,d),n]
 *   (E4) C'[p,n]   = sum R[m,k] T'[m,r,p] Q[(k,r),n]          (Fig. 1(f), 3rd diagram)
 *   then C <- sym(C')/||.||_F, T <- sym(T')/||.||_F.
 * A NaN/Inf/zero norm is reported by the next synchronising call. */
int qrctm_step(qrctm_t* h);

/* Iterate: step; every CHECK_EVERY steps compute s = descending |eigenvalues|
 * of C and delta = max_i |s_i - s_i(previous check)|; stop when delta < tol or
 * after max_iter steps.  Synchronises before returning.  iters_done = steps
 * executed; final_delta = last delta (+inf if never checked).  Either output
 * pointer may be NULL.  HOST pointers. */
int qrctm_run(qrctm_t* h, int max_iter, double tol, int* iters_done, double* final_delta);

/* Copy the current normalised environment out (either pointer may be NULL). */
int qrctm_get_env(qrctm_t* h, double* C, double* T);

/* Descending singular values (= |eigenvalues|) of the current normalised C,
 * computed on the device (Householder tridiagonalisation + Sturm bisection); s has chi
 * entries; sum s^2 = 1. */
int qrctm_get_corner_spectrum(qrctm_t* h, double* s);

/* Q[chi*b][chi] and R[chi][chi] of the last step (either may be NULL). */
int qrctm_get_qr(qrctm_t* h, double* Q, double* R);

/* Un-normalised C'[chi][chi], T'[chi][b][chi] of the last step (either may be NULL). */
int qrctm_get_raw(qrctm_t* h, double* Cn, double* Tn);

/* Copy the double-layer tensor a[b][b][b][b] out. */
int qrctm_get_a(qrctm_t* h, double* a);

/* Norm per site kappa = Z1 * Z4 / Z2^2 of the current environment, with
 * Z4 = tr C^4, Z2 the 2x3 network CTC/CTC, Z1 the 3x3 network CTC/TaT/CTC
 * (reading A8).  HOST pointer.  Synchronises. */
int qrctm_norm_per_site(qrctm_t* h, double* kappa);

/* NEXT-3.  Expectation value of a two-site operator on a nearest-neighbour bond,
 *   e_bond = Tr(rho2 H) / Tr(rho2),   rho2[s1,s1',s2,s2'] = sum LH^{s1 s1'}[k,x,k'] LH^{s2 s2'}[k,x,k'],
 * LH^{ss'} = (E3) with c~ = C.T in place of Q and a^{ss'} = A[s] (x) A[s'] in place of a  (the left half of the network
 * C T T C / T a a T / C T T C; the right half is its mirror image under C4v).  H is d^2 x d^2 row-major with index
 * [(s1 s2)][(s1' s2')] (HOST).  The energy per site of H_total = sum_<ij> h_ij on the square lattice is 2 e_bond
 * (PAPER.md:38-40).  rho_out (HOST, d^4, may be NULL) receives the un-normalised rho2.  d <= 4.  Overwrites the
 * step scratch (X, P, S); the environment is untouched.  Synchronises. */
int qrctm_energy_nn(qrctm_t* h, const double* H, double* e_bond, double* rho_out);

/* K3 -> K4 -> K5 alone (the edge renormalisation of PAPER.md:32, "T' = Q^T (T a) Q"), with an arbitrary matrix U
 * in place of Q:  Tout[m][r][n] = sum U[(j,u),m] T[j,l,J] a[u,l,d,r] U[(J,d),n]   (E3)
 * U[chi*b][ncols] row-major (HOST or DEVICE), 1 <= ncols <= chi capacity; Tout[ncols][b][ncols] (HOST or DEVICE).
 * Uses the current T and a; overwrites the step scratch (P, S); the environment is untouched.  Synchronises.
 * For the sub-step parity tests (an isometry that is not a QR factor). */
int qrctm_edge_update(qrctm_t* h, const double* U, int ncols, double* Tout);

/* min_k R_kk / max_k R_kk of the last step: a conditioning diagnostic for the
 * uniqueness of Q (DESIGN.md hazard H1).  HOST pointer.  Synchronises. */
int qrctm_r_diag_ratio(qrctm_t* h, double* ratio);

int qrctm_set_option(qrctm_t* h, int key, int value);

/* Number of kernels this handle has launched so far (for bench.py's
 * gpu_launches); kernels replayed from a CUDA graph are counted per replay. */
long long qrctm_launch_count(const qrctm_t* h);

/* Per-iteration history of the current environment (reset by qrctm_set_env / qrctm_init_bulk / qrctm_eig_step), kept on the device
 * in a ring buffer of 4096 records and written by the step's own kernels (K7, K8) -- nothing is logged on the hot
 * path.  Record i (4 doubles): delta_i = max_k |s_k - s_k(previous check)| (NaN if that step was not checked),
 * ||C'||_F and ||T'||_F before normalisation, min_k R_kk / max_k R_kk of the step's QR (hazard H1).
 * *n_steps = iterations recorded since the reset; out (HOST, 4 * max_records doubles) receives the last
 * min(n_steps, max_records, 4096) records in chronological order.  Synchronises. */
int qrctm_get_history(qrctm_t* h, double* out, int max_records, int* n_steps);

/* Event-timed profile of one step: runs one qrctm_step with CUDA events around
 * each stage and returns milliseconds in ms[0..QRCTM_NSTAGE-1]:
 * 0 K1 reduced corner, 1 K2 QR (panel+WY+form Q+sign), 2 K3 half-absorb,
 * 3 K4 absorb a, 4 K5 project, 5 K6 corner, 6 K7 symmetrise+normalise. */
#define QRCTM_NSTAGE 7
int qrctm_profile_step(qrctm_t* h, float* ms);

/* Per-stage device time accumulated by qrctm_run while QRCTM_OPT_TIME_STAGES = 1:
 * ms[0..6] as in qrctm_profile_step, ms[7] = K8 spectrum + delta; *steps = number
 * of steps accumulated.  reset != 0 clears the accumulators.  HOST pointers. */
int qrctm_get_stage_ms(qrctm_t* h, double* ms /* QRCTM_NSTAGE + 1 */, long long* steps, int reset);

/* Stand-alone FP64 GEMM entry used by the sub-step parity tests and the
 * roofline bench:  Cmat[M][N] = op(A) * B with B[K][N] row-major and
 * op(A) = A[M][K] (transA = 0) or A stored as [K][M] (transA = 1).
 * DEVICE pointers, leading dimensions in elements. path: see QRCTM_OPT_GEMM_PATH. */
int qrctm_gemm_f64(void* cuda_stream, int path, int transA, int M, int N, int K,
                   const double* A, long long lda, const double* B, long long ldb,
                   double* Cmat, long long ldc);
/* The same with a scratch buffer: work (DEVICE, work_bytes bytes, 16-byte aligned, may be NULL / 0) lets the
 * launcher use its K-splitting schedules - split-K with a fixed-order reduction, and stream-K for GEMMs whose tiles
 * fill only a few ragged waves - exactly as the stages of qrctm_step do with the handle's
 * workspace.  The result does not depend on the schedule beyond the summation order (<= 1e-13 relative). */
int qrctm_gemm_f64_ws(void* cuda_stream, int path, int transA, int M, int N, int K,
                      const double* A, long long lda, const double* B, long long ldb,
                      double* Cmat, long long ldc, void* work, unsigned long long work_bytes);

/* The same GEMM for callers that cannot allocate (code under CUDA-graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): Cmat[M][N] = op(A) * B as qrctm_gemm_f64_ws (DMMA path), but the K-splitting scratch (split-K
 * partial outputs / stream-K partial tiles) is a file-scope device array inside the library -- 16 MiB on every GPU
 * that loads libqrctm.so, held until the process exits.  The call itself allocates nothing (no cudaMalloc / cudaFree,
 * no allocating library routine); inputs and the output are the caller's DEVICE buffers.
 * Limit: M * N <= 65536 (e.g. the chi x chi Gram and corner products with long K); larger shapes are rejected with
 * QRCTM_ERR_INVALID_ARG and a text in qrctm_noalloc_last_error() (thread-local; empty after a successful call).
 * The scratch is SHARED by every call on that GPU and keeps the last call's contents: nothing in it has to start at
 * zero (every partial the reduction reads is written by the same call first), but two calls that overlap on the GPU
 * (different streams, or graphs replayed concurrently) race on it -- serialise them. */
int qrctm_gemm_f64_noalloc(void* cuda_stream, int transA, int M, int N, int K, const double* A, long long lda,
                           const double* B, long long ldb, double* Cmat, long long ldc);
const char* qrctm_noalloc_last_error(void);

/* Stand-alone QR entry (K2): factor X[rows][cols] (DEVICE, row-major, cols <=
 * rows) into Q[rows][cols], R[cols][cols] with diag(R) >= 0 (path: see
 * QRCTM_OPT_QR_PATH; path 0 synchronises the stream once to read the device-side accuracy verdict). work must hold
 * qrctm_qr_work_bytes(rows, cols) bytes (DEVICE). */
unsigned long long qrctm_qr_work_bytes(int rows, int cols);
int qrctm_qr_f64(void* cuda_stream, int path, int rows, int cols, const double* X, double* Q,
                 double* R, void* work);

/* Stand-alone entry of the n x n factorisation inside CholeskyQR2 (K2, csrc/cholqr.cuh; for the sub-step parity
 * tests): G[n][n] symmetric positive definite (DEVICE; its lower triangle is read), n <= 208.
 *   R[n][n]    = chol(G)^T, upper triangular (G = R^T R), zeros below the diagonal            (DEVICE)
 *   Rinv[n][n] = R^-1, upper triangular                                                       (DEVICE)
 *   status[0]  = 1 if a pivot was not positive and finite (the factor is then meaningless)    (DEVICE int)
 *   dev[0]     = ||G - I||_F                                                                  (DEVICE)
 *   prof       = NULL, or 8 DEVICE long longs: SM cycles of the kernel's phases (load; diagonal blocks; panels;
 *                trailing updates; write R; diagonal-block inverses; inverse; write R^-1).
 * One CTA; asynchronous on the stream. */
int qrctm_chol_inv_f64(void* cuda_stream, int n, const double* G, double* R, double* Rinv, int* status, double* dev,
                       long long* prof);

/* Stand-alone entry of K8's tridiagonalisation (csrc/spectrum.cuh; for the sub-step parity tests): the symmetric
 * C[n][n] (DEVICE; lower triangle read, untouched), n <= 216, is reduced by Householder similarity transforms to the
 * tridiagonal matrix with diagonal d[n] and sub-diagonal e[1..n-1] (e[0] = 0) (DEVICE).  prof = NULL, or 8 DEVICE
 * long longs: SM cycles of the kernel's phases.  One CTA; asynchronous on the stream. */
int qrctm_tridiag_f64(void* cuda_stream, int n, const double* C, double* d, double* e, long long* prof);

/* ---- NEXT-2: the paper's initialisation and warm-up ----
 * PAPER.md:28 "performing only a few (1-4) initial warm-up steps using the standard
 * CTMRG scheme is sufficient. This warm-up phase also enables chi to be dynamically
 * increased up to the desired target value."; the initial boundary from the bulk
 * tensors is fn.[48].
 *
 * qrctm_get_chi: the CURRENT environment bond dimension (below the capacity the
 *   handle was created with only between qrctm_init_bulk and the end of the
 *   warm-up) and that capacity.  Either pointer may be NULL.  HOST pointers.
 * qrctm_init_bulk: C0[(d d'),(r r')] = sum_{s,u,l} A A, T0[(l l'),(d d'),(r r')] =
 *   sum_{s,u} A A (fn.[48]), normalised (K7); the current chi becomes D^2.
 *   Needs set_A; QRCTM_ERR_INVALID_ARG if D^2 > capacity.
 * qrctm_eig_step: one standard CTMRG iteration (Fig. 1(d)):
 *   C~ (E5) from the current C, T; its chi_new eigenpairs of largest |lambda|
 *   (ties: ascending eigenvalue order first, reading A9) -> U, sign gauge
 *   "largest-magnitude component of every column positive"; C' = diag(lambda),
 *   T' = (E3) with U for Q; K7.  chi_new = 0 keeps chi; otherwise
 *   1 <= chi_new <= min(capacity, chi D^2).  The eigensolver is the library's own
 *   (Householder tridiagonalisation, multisection, inverse iteration; csrc/eigh.cuh)
 *   and needs chi D^2 <= 14000; its workspace is a separate DEVICE allocation owned
 *   by the handle, made on first use.  The next qrctm_run starts a fresh convergence
 *   history (s_prev = spectrum of the new C).
 * qrctm_get_eig: U (rows x cols, row-major) and lambda (cols) of the last
 *   qrctm_eig_step; rows/cols (HOST, may be NULL) are always written, U / lam
 *   (HOST or DEVICE, may be NULL) only if non-NULL.  QRCTM_ERR_NOT_READY before
 *   the first eigen step.
 * qrctm_warmup: qrctm_init_bulk, then n_eig_steps eigen steps with
 *   chi <- min(capacity, chi D^2) each. */
int qrctm_get_chi(const qrctm_t* h, int* chi, int* chi_capacity);
int qrctm_init_bulk(qrctm_t* h);
int qrctm_eig_step(qrctm_t* h, int chi_new);
int qrctm_get_eig(qrctm_t* h, double* U, double* lam, int* rows, int* cols);
int qrctm_warmup(qrctm_t* h, int n_eig_steps);

/* Stand-alone entry of the eigensolver used by qrctm_eig_step: the k eigenpairs of
 * largest |lambda| of the symmetric A[n][n] (DEVICE, row-major, DESTROYED):
 * lam[k] (DEVICE) in decreasing |lambda| (ties: the smaller eigenvalue first),
 * U[n][k] (DEVICE, row-major) orthonormal, largest-magnitude component of each
 * column positive.  1 <= k <= n <= 14000.  work: qrctm_eigh_work_bytes(n, k) bytes
 * (DEVICE); 0 is returned for unsupported sizes. */
unsigned long long qrctm_eigh_work_bytes(int n, int k);
int qrctm_eigh_top_f64(void* cuda_stream, int n, int k, double* A, double* lam, double* U, void* work);

/* ---- NEXT-4 ("the use of multiple GPUs") ----
 * One iteration sharded over the column index m of Q: K3 -> K4 -> K5 never mix different m
 * (P[:,m,:,:], S[m,...], T'[m,:,:]), and (E4) is a sum over m.  Every rank holds the same
 * A, C, T (replicated, as is the cheap K1 + K2), computes the rows m in [m0, m1) of T' and
 * its partial C', and ONE exchange step assembles them: all-gather of the T' slices
 * (8 chi^2 D^2 bytes in total), all-reduce of the partial C' (8 chi^2 bytes).  The library
 * does not link a communication library: the exchange is done by the caller on the DEVICE
 * buffers qrctm_shard_buffers returns (the Python binding uses torch.distributed / NCCL).
 *
 * qrctm_shard_range: this rank's contiguous range [m0, m1) of m (sizes differ by <= 1;
 *   empty when nranks > chi).  HOST pointers.
 * qrctm_shard_front: K1, K2, then K3-K5 and the partial (E4) for this rank's range.
 *   Afterwards Tn (chi x D^2 x chi, rows m) holds this rank's rows and ZEROS elsewhere,
 *   Cn (chi x chi) the partial corner -- so either an all-gather of the row blocks or a
 *   plain sum over ranks of the whole buffers assembles T' and C'.  nranks = 1 gives the
 *   un-normalised result of an ordinary step.
 * qrctm_shard_buffers: DEVICE pointers of Cn and Tn inside the handle's workspace
 *   (owned by the handle; valid until qrctm_destroy).
 * qrctm_shard_finish: K7 on the exchanged Cn, Tn -> the new C, T.  The caller must order
 *   the exchange before it on the handle's stream. */
int qrctm_shard_range(int chi, int rank, int nranks, int* m0, int* m1);
int qrctm_shard_front(qrctm_t* h, int rank, int nranks);
int qrctm_shard_buffers(qrctm_t* h, double** Cn, double** Tn);
int qrctm_shard_finish(qrctm_t* h);

/* FP64 issue-rate probe (roofline denominators):
 * kind 0 = DFMA chains, 1 = DMMA m8n8k4 chains.  Returns TFLOP/s measured with
 * CUDA events over `iters` loop trips on every SM.  HOST pointer. */
int qrctm_probe_fp64(int kind, int iters, double* tflops);

const char* qrctm_last_error(const qrctm_t* h);
const char* qrctm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QRCTM_H */
