"""Thin Python binding of libqrctm.so (include/qrctm.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the shared library; this
module allocates device memory through PyTorch, passes raw pointers and the
current CUDA stream, and turns status codes into exceptions.  There is NO CPU
fallback: if the library is missing or no CUDA device is present the calls
raise.  Names follow include/qrctm.h one to one.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import (POINTER, byref, c_char_p, c_double, c_float, c_int, c_longlong, c_ulonglong,
                    c_void_p)

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("QRCTM_LIB", os.path.join(_HERE, "libqrctm.so"))

QRCTM_OK = 0
OPT_CORNER_MODE, OPT_SYMMETRIZE, OPT_CHECK_EVERY, OPT_GEMM_PATH, OPT_TIME_STAGES, OPT_QR_PATH, OPT_OVERLAP_CHECK, OPT_USE_GRAPH, OPT_ABSORB_MODE, OPT_K8_PATH, OPT_SMALL_PATH = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11
NSTAGE = 7
STAGE_NAMES = ("K1_reduced_corner", "K2_qr", "K3_half_absorb", "K4_absorb_a", "K5_project",
               "K6_corner", "K7_normalize")
STAGE_NAMES_RUN = STAGE_NAMES + ("K8_spectrum",)

# every symbol include/qrctm.h declares (tests check that the .so exports them all)
SYMBOLS = (
    "qrctm_create", "qrctm_workspace_bytes", "qrctm_create_in", "qrctm_destroy", "qrctm_set_stream",
    "qrctm_set_A", "qrctm_set_env", "qrctm_step", "qrctm_run", "qrctm_get_env",
    "qrctm_get_corner_spectrum", "qrctm_get_qr", "qrctm_get_raw", "qrctm_get_a", "qrctm_norm_per_site",
    "qrctm_r_diag_ratio", "qrctm_energy_nn", "qrctm_edge_update", "qrctm_set_option", "qrctm_launch_count", "qrctm_get_history", "qrctm_get_stage_ms", "qrctm_profile_step",
    "qrctm_gemm_f64", "qrctm_gemm_f64_ws", "qrctm_gemm_f64_noalloc", "qrctm_noalloc_last_error", "qrctm_qr_work_bytes", "qrctm_qr_f64", "qrctm_probe_fp64", "qrctm_last_error",
    "qrctm_version",
    "qrctm_get_chi", "qrctm_init_bulk", "qrctm_eig_step", "qrctm_get_eig", "qrctm_warmup",
    "qrctm_eigh_work_bytes", "qrctm_eigh_top_f64", "qrctm_chol_inv_f64", "qrctm_tridiag_f64",
    "qrctm_shard_range", "qrctm_shard_front", "qrctm_shard_buffers", "qrctm_shard_finish",
)


class QrctmError(RuntimeError):
    pass


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libqrctm.so (built in-tree by __graft_entry__.build()).  Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise QrctmError(f"{LIB_PATH} not found: run `python -c 'import __graft_entry__ as g; g.build()'` "
                         "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    P = c_void_p
    lib.qrctm_create.argtypes = [c_int, c_int, c_int, POINTER(P)]
    lib.qrctm_workspace_bytes.argtypes = [c_int, c_int, c_int]
    lib.qrctm_workspace_bytes.restype = c_ulonglong
    lib.qrctm_create_in.argtypes = [c_int, c_int, c_int, P, c_ulonglong, POINTER(P)]
    lib.qrctm_destroy.argtypes = [P]
    lib.qrctm_set_stream.argtypes = [P, P]
    lib.qrctm_set_A.argtypes = [P, P]
    lib.qrctm_set_env.argtypes = [P, P, P]
    lib.qrctm_step.argtypes = [P]
    lib.qrctm_run.argtypes = [P, c_int, c_double, POINTER(c_int), POINTER(c_double)]
    lib.qrctm_get_env.argtypes = [P, P, P]
    lib.qrctm_get_corner_spectrum.argtypes = [P, P]
    lib.qrctm_get_qr.argtypes = [P, P, P]
    lib.qrctm_get_raw.argtypes = [P, P, P]
    lib.qrctm_get_a.argtypes = [P, P]
    lib.qrctm_norm_per_site.argtypes = [P, POINTER(c_double)]
    lib.qrctm_r_diag_ratio.argtypes = [P, POINTER(c_double)]
    lib.qrctm_energy_nn.argtypes = [P, P, POINTER(c_double), P]
    lib.qrctm_edge_update.argtypes = [P, P, c_int, P]
    lib.qrctm_get_history.argtypes = [P, P, c_int, POINTER(c_int)]
    lib.qrctm_set_option.argtypes = [P, c_int, c_int]
    lib.qrctm_launch_count.argtypes = [P]
    lib.qrctm_launch_count.restype = c_longlong
    lib.qrctm_profile_step.argtypes = [P, POINTER(c_float)]
    lib.qrctm_get_stage_ms.argtypes = [P, POINTER(c_double), POINTER(c_longlong), c_int]
    lib.qrctm_gemm_f64.argtypes = [P, c_int, c_int, c_int, c_int, c_int, P, c_longlong, P, c_longlong, P,
                                   c_longlong]
    lib.qrctm_gemm_f64_ws.argtypes = [P, c_int, c_int, c_int, c_int, c_int, P, c_longlong, P, c_longlong, P,
                                      c_longlong, P, c_ulonglong]
    lib.qrctm_gemm_f64_noalloc.argtypes = [P, c_int, c_int, c_int, c_int, P, c_longlong, P, c_longlong, P, c_longlong]
    lib.qrctm_noalloc_last_error.restype = c_char_p
    lib.qrctm_qr_work_bytes.argtypes = [c_int, c_int]
    lib.qrctm_qr_work_bytes.restype = c_ulonglong
    lib.qrctm_qr_f64.argtypes = [P, c_int, c_int, c_int, P, P, P, P]
    lib.qrctm_probe_fp64.argtypes = [c_int, c_int, POINTER(c_double)]
    lib.qrctm_chol_inv_f64.argtypes = [P, c_int, P, P, P, P, P, P]
    lib.qrctm_tridiag_f64.argtypes = [P, c_int, P, P, P, P]
    lib.qrctm_get_chi.argtypes = [P, POINTER(c_int), POINTER(c_int)]
    lib.qrctm_init_bulk.argtypes = [P]
    lib.qrctm_eig_step.argtypes = [P, c_int]
    lib.qrctm_get_eig.argtypes = [P, P, P, POINTER(c_int), POINTER(c_int)]
    lib.qrctm_warmup.argtypes = [P, c_int]
    lib.qrctm_eigh_work_bytes.argtypes = [c_int, c_int]
    lib.qrctm_eigh_work_bytes.restype = c_ulonglong
    lib.qrctm_eigh_top_f64.argtypes = [P, c_int, c_int, P, P, P, P]
    lib.qrctm_shard_range.argtypes = [c_int, c_int, c_int, POINTER(c_int), POINTER(c_int)]
    lib.qrctm_shard_front.argtypes = [P, c_int, c_int]
    lib.qrctm_shard_buffers.argtypes = [P, POINTER(P), POINTER(P)]
    lib.qrctm_shard_finish.argtypes = [P]
    lib.qrctm_last_error.argtypes = [P]
    lib.qrctm_last_error.restype = c_char_p
    lib.qrctm_version.restype = c_char_p
    _lib = lib
    return lib


def _ptr(x):
    """Raw pointer of a numpy array (host) or torch tensor (host or device)."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        if x.dtype != np.float64 or not x.flags["C_CONTIGUOUS"]:
            raise QrctmError("numpy arguments must be C-contiguous float64")
        return x.ctypes.data_as(c_void_p)
    import torch
    if isinstance(x, torch.Tensor):
        if x.dtype != torch.float64 or not x.is_contiguous():
            raise QrctmError("torch arguments must be contiguous float64")
        return c_void_p(x.data_ptr())
    raise QrctmError(f"unsupported argument type {type(x)}")


class QRCTM:
    """Handle of one (d, D, chi) QR-CTMRG problem on the current CUDA device.

    Device workspace is a torch uint8 tensor (PyTorch owns device memory); work is
    enqueued on `self.stream`, a torch.cuda.Stream owned by the handle (a non-default
    stream, so that the library can capture the step into CUDA graphs).  Calls that take
    device tensors first make that stream wait for the caller's current stream; every
    get_* / run / norm_per_site call synchronises before returning.
    """

    def __init__(self, d: int, D: int, chi: int, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise QrctmError("no CUDA device: the QR-CTMRG path has no CPU fallback")
        self.lib = load_library()
        self.d, self.D, self.chi_cap, self.b = d, D, chi, D * D      # self.chi: the current chi (property)
        nbytes = self.lib.qrctm_workspace_bytes(d, D, chi)
        if nbytes == 0:
            raise QrctmError("invalid (d, D, chi)")
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        base = (self._ws.data_ptr() + 255) // 256 * 256
        h = c_void_p()
        rc = self.lib.qrctm_create_in(d, D, chi, c_void_p(base), nbytes, byref(h))
        if rc != QRCTM_OK:
            raise QrctmError(f"qrctm_create_in failed: {rc}")
        self._h = h
        self.stream = stream if stream is not None else torch.cuda.Stream()
        self.stream.wait_stream(torch.cuda.current_stream())
        self._check(self.lib.qrctm_set_stream(h, c_void_p(self.stream.cuda_stream)))

    @property
    def chi(self) -> int:
        """Current environment bond dimension (== the capacity except during the NEXT-2 warm-up)."""
        c = c_int(0)
        self._check(self.lib.qrctm_get_chi(self._h, byref(c), None))
        return c.value

    # -- plumbing
    def _check(self, rc: int):
        if rc != QRCTM_OK:
            msg = self.lib.qrctm_last_error(self._h)
            raise QrctmError(f"qrctm error {rc}: {msg.decode() if msg else ''}")

    def close(self):
        if getattr(self, "_h", None):
            self.lib.qrctm_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _out(self, shape, like_device: bool):
        if like_device:
            import torch
            return torch.empty(shape, dtype=torch.float64, device="cuda")
        return np.empty(shape, dtype=np.float64)

    # -- the C ABI, same names
    def set_stream(self, stream):
        """stream: a torch.cuda.Stream"""
        self.stream = stream
        self._check(self.lib.qrctm_set_stream(self._h, c_void_p(stream.cuda_stream)))

    def synchronize(self):
        self.stream.synchronize()

    def _order_after_caller(self, *tensors):
        """The handle's stream waits for the caller's current stream; torch CUDA inputs are recorded on the handle's
        stream, so that the caching allocator does not reuse them while an asynchronous copy is still pending."""
        import torch
        self.stream.wait_stream(torch.cuda.current_stream())
        for t in tensors:
            if isinstance(t, torch.Tensor) and t.is_cuda:
                t.record_stream(self.stream)

    def set_A(self, A):
        assert tuple(A.shape) == (self.d,) + (self.D,) * 4
        self._order_after_caller(A)
        self._check(self.lib.qrctm_set_A(self._h, _ptr(A)))

    def set_env(self, C, T):
        n = self.chi_cap
        assert tuple(C.shape) == (n, n) and tuple(T.shape) == (n, self.b, n)
        self._order_after_caller(C, T)
        self._check(self.lib.qrctm_set_env(self._h, _ptr(C), _ptr(T)))

    def step(self):
        self._check(self.lib.qrctm_step(self._h))

    def run(self, max_iter: int, tol: float):
        it, dl = c_int(0), c_double(0.0)
        self._check(self.lib.qrctm_run(self._h, max_iter, tol, byref(it), byref(dl)))
        return it.value, dl.value

    def get_env(self, device: bool = False):
        n = self.chi
        C = self._out((n, n), device)
        T = self._out((n, self.b, n), device)
        self._check(self.lib.qrctm_get_env(self._h, _ptr(C), _ptr(T)))
        return C, T

    def get_corner_spectrum(self):
        s = np.empty(self.chi, dtype=np.float64)
        self._check(self.lib.qrctm_get_corner_spectrum(self._h, _ptr(s)))
        return s

    def get_qr(self, device: bool = False):
        n = self.chi
        Q = self._out((n * self.b, n), device)
        R = self._out((n, n), device)
        self._check(self.lib.qrctm_get_qr(self._h, _ptr(Q), _ptr(R)))
        return Q, R

    def get_raw(self, device: bool = False):
        n = self.chi
        Cn = self._out((n, n), device)
        Tn = self._out((n, self.b, n), device)
        self._check(self.lib.qrctm_get_raw(self._h, _ptr(Cn), _ptr(Tn)))
        return Cn, Tn

    def init_bulk(self):
        self._check(self.lib.qrctm_init_bulk(self._h))

    def eig_step(self, chi_new: int = 0):
        self._check(self.lib.qrctm_eig_step(self._h, chi_new))

    def get_eig(self, device: bool = False):
        r, c = c_int(0), c_int(0)
        self._check(self.lib.qrctm_get_eig(self._h, None, None, byref(r), byref(c)))
        U = self._out((r.value, c.value), device)
        lam = self._out((c.value,), device)
        self._check(self.lib.qrctm_get_eig(self._h, _ptr(U), _ptr(lam), None, None))
        return U, lam

    def warmup(self, n_eig_steps: int):
        self._check(self.lib.qrctm_warmup(self._h, n_eig_steps))

    # -- NEXT-4: one iteration sharded over ranks (one process per GPU)
    def shard_front(self, rank: int, nranks: int):
        self._check(self.lib.qrctm_shard_front(self._h, rank, nranks))

    def shard_buffers(self):
        """(Cn, Tn): torch views of the handle's device buffers the exchange works on."""
        import torch
        pc, pt = c_void_p(), c_void_p()
        self._check(self.lib.qrctm_shard_buffers(self._h, byref(pc), byref(pt)))
        n, base = self.chi, self._ws.data_ptr()

        def view(ptr, count, shape):
            off = ptr - base
            return self._ws[off:off + 8 * count].view(torch.float64).view(shape)
        return view(pc.value, n * n, (n, n)), view(pt.value, n * self.b * n, (n, self.b * n))

    def shard_finish(self):
        self._check(self.lib.qrctm_shard_finish(self._h))

    def shard_step(self, rank: int, nranks: int, group=None):
        """One QR-CTMRG iteration with K3-K5 split over `nranks` processes (torch.distributed must be initialised
        when nranks > 1); every rank ends with the same new C, T."""
        import torch
        self.shard_front(rank, nranks)
        if nranks > 1:
            Cn, Tn = self.shard_buffers()
            with torch.cuda.stream(self.stream):
                shard_exchange(Cn, Tn, rank, nranks, group)
        self.shard_finish()

    def get_a(self):
        a = np.empty((self.b,) * 4, dtype=np.float64)
        self._check(self.lib.qrctm_get_a(self._h, _ptr(a)))
        return a

    def norm_per_site(self) -> float:
        k = c_double(0.0)
        self._check(self.lib.qrctm_norm_per_site(self._h, byref(k)))
        return k.value

    def energy_nn(self, H, return_rho: bool = False):
        """Tr(rho2 H)/Tr(rho2) on a nearest-neighbour bond; H is (d*d, d*d) with index [(s1 s2), (s1' s2')]."""
        H = np.ascontiguousarray(H, dtype=np.float64)
        assert H.shape == (self.d * self.d, self.d * self.d)
        e = c_double(0.0)
        rho = np.empty((self.d,) * 4, dtype=np.float64) if return_rho else None
        self._check(self.lib.qrctm_energy_nn(self._h, _ptr(H), byref(e), _ptr(rho)))
        return (e.value, rho) if return_rho else e.value

    def edge_update(self, U, device: bool = False):
        """T' = (E3) with the (chi*b, n) matrix U in place of Q, from the current T and a."""
        n = int(U.shape[1])
        assert int(U.shape[0]) == self.chi * self.b
        self._order_after_caller(U)
        out = self._out((n, self.b, n), device)
        self._check(self.lib.qrctm_edge_update(self._h, _ptr(U), n, _ptr(out)))
        return out

    def r_diag_ratio(self) -> float:
        k = c_double(0.0)
        self._check(self.lib.qrctm_r_diag_ratio(self._h, byref(k)))
        return k.value

    def set_option(self, key: int, value: int):
        self._check(self.lib.qrctm_set_option(self._h, key, value))

    def get_history(self, max_records: int = 4096):
        """(records, n_steps): records[i] = (delta, ||C'||_F, ||T'||_F, min R_kk / max R_kk) of the last iterations."""
        out = np.empty((max(max_records, 1), 4), dtype=np.float64)
        n = c_int(0)
        self._check(self.lib.qrctm_get_history(self._h, _ptr(out), max_records, byref(n)))
        return out[:min(n.value, max_records, 4096)].copy(), n.value

    def launch_count(self) -> int:
        return int(self.lib.qrctm_launch_count(self._h))

    def get_stage_ms(self, reset: bool = False):
        """(dict stage -> total ms, steps) accumulated by run() while OPT_TIME_STAGES = 1."""
        ms = (c_double * (NSTAGE + 1))()
        n = c_longlong(0)
        self._check(self.lib.qrctm_get_stage_ms(self._h, ms, byref(n), int(reset)))
        return dict(zip(STAGE_NAMES_RUN, [float(x) for x in ms])), int(n.value)

    def profile_step(self):
        ms = (c_float * NSTAGE)()
        self._check(self.lib.qrctm_profile_step(self._h, ms))
        return dict(zip(STAGE_NAMES, [float(x) for x in ms]))


# -- stand-alone entries (device tensors in, device tensors out)
def gemm_f64(A, B, transA: bool = False, path: int = 0, work_bytes: int = 0):
    """out[M,N] = op(A) @ B on the GPU through qrctm_gemm_f64 (torch CUDA float64 tensors);
    work_bytes > 0: through qrctm_gemm_f64_ws with a scratch buffer of that size (split-K / stream-K schedules)."""
    import torch
    lib = load_library()
    K, N = B.shape
    M = A.shape[1] if transA else A.shape[0]
    assert (A.shape[0] if transA else A.shape[1]) == K
    for t in (A, B):       # row-strided views are fine: the ABI takes leading dimensions
        if t.dtype != torch.float64 or not t.is_cuda or t.stride(1) != 1:
            raise QrctmError("gemm_f64 wants CUDA float64 matrices with unit column stride")
    out = torch.empty((M, N), dtype=torch.float64, device="cuda")
    if work_bytes > 0:
        work = torch.empty(work_bytes, dtype=torch.uint8, device="cuda")
        rc = lib.qrctm_gemm_f64_ws(c_void_p(torch.cuda.current_stream().cuda_stream), path, int(transA), M, N, K,
                                   c_void_p(A.data_ptr()), A.stride(0), c_void_p(B.data_ptr()), B.stride(0),
                                   _ptr(out), N, c_void_p(work.data_ptr()), work_bytes)
    else:
        rc = lib.qrctm_gemm_f64(c_void_p(torch.cuda.current_stream().cuda_stream), path, int(transA), M, N, K,
                                c_void_p(A.data_ptr()), A.stride(0), c_void_p(B.data_ptr()), B.stride(0),
                                _ptr(out), N)
    if rc != QRCTM_OK:
        raise QrctmError(f"qrctm_gemm_f64 failed: {rc}")
    return out


def gemm_f64_noalloc(A, B, out, transA: bool = False):
    """out[M,N] = op(A) @ B through qrctm_gemm_f64_noalloc: the library allocates nothing (static device scratch);
    `out` is the caller's CUDA float64 tensor.  M * N <= 65536."""
    import torch
    lib = load_library()
    K, N = B.shape
    M = A.shape[1] if transA else A.shape[0]
    assert (A.shape[0] if transA else A.shape[1]) == K and tuple(out.shape) == (M, N)
    for t in (A, B, out):
        if t.dtype != torch.float64 or not t.is_cuda or t.stride(1) != 1:
            raise QrctmError("gemm_f64_noalloc wants CUDA float64 matrices with unit column stride")
    rc = lib.qrctm_gemm_f64_noalloc(c_void_p(torch.cuda.current_stream().cuda_stream), int(transA), M, N, K,
                                    c_void_p(A.data_ptr()), A.stride(0), c_void_p(B.data_ptr()), B.stride(0),
                                    c_void_p(out.data_ptr()), out.stride(0))
    if rc != QRCTM_OK:
        raise QrctmError(f"qrctm_gemm_f64_noalloc failed ({rc}): {lib.qrctm_noalloc_last_error().decode()}")
    return out


def qr_f64(X, path: int = 0):
    """(Q, R) with diag(R) >= 0 of a torch CUDA float64 matrix through qrctm_qr_f64."""
    import torch
    lib = load_library()
    rows, cols = X.shape
    Q = torch.empty((rows, cols), dtype=torch.float64, device="cuda")
    R = torch.empty((cols, cols), dtype=torch.float64, device="cuda")
    work = torch.empty(lib.qrctm_qr_work_bytes(rows, cols), dtype=torch.uint8, device="cuda")
    rc = lib.qrctm_qr_f64(c_void_p(torch.cuda.current_stream().cuda_stream), path, rows, cols, _ptr(X), _ptr(Q),
                          _ptr(R), c_void_p(work.data_ptr()))
    if rc != QRCTM_OK:
        raise QrctmError(f"qrctm_qr_f64 failed: {rc}")
    torch.cuda.current_stream().synchronize()
    return Q, R


def chol_inv_f64(G, profile: bool = False):
    """(R, Rinv, status, dev[, cycles]) of a symmetric positive definite torch CUDA float64 matrix (n <= 208) through
    qrctm_chol_inv_f64: G = R^T R with R upper triangular."""
    import torch
    lib = load_library()
    n = G.shape[0]
    R = torch.empty((n, n), dtype=torch.float64, device="cuda")
    Ri = torch.empty((n, n), dtype=torch.float64, device="cuda")
    st = torch.zeros(1, dtype=torch.int32, device="cuda")
    dev = torch.zeros(1, dtype=torch.float64, device="cuda")
    prof = torch.zeros(8, dtype=torch.int64, device="cuda") if profile else None
    rc = lib.qrctm_chol_inv_f64(c_void_p(torch.cuda.current_stream().cuda_stream), n, _ptr(G.contiguous()), _ptr(R), _ptr(Ri),
                                c_void_p(st.data_ptr()), _ptr(dev), c_void_p(prof.data_ptr()) if profile else None)
    if rc != QRCTM_OK:
        raise QrctmError(f"qrctm_chol_inv_f64 failed: {rc}")
    torch.cuda.current_stream().synchronize()
    out = (R, Ri, int(st.item()), float(dev.item()))
    return out + (prof.cpu().numpy(),) if profile else out


def tridiag_f64(C, profile: bool = False):
    """(d, e[, cycles]) of a symmetric torch CUDA float64 matrix (n <= 216) through qrctm_tridiag_f64."""
    import torch
    lib = load_library()
    n = C.shape[0]
    d = torch.empty((n,), dtype=torch.float64, device="cuda")
    e = torch.empty((n,), dtype=torch.float64, device="cuda")
    prof = torch.zeros(8, dtype=torch.int64, device="cuda") if profile else None
    rc = lib.qrctm_tridiag_f64(c_void_p(torch.cuda.current_stream().cuda_stream), n, _ptr(C.contiguous()), _ptr(d), _ptr(e),
                               c_void_p(prof.data_ptr()) if profile else None)
    if rc != QRCTM_OK:
        raise QrctmError(f"qrctm_tridiag_f64 failed: {rc}")
    torch.cuda.current_stream().synchronize()
    return (d, e, prof.cpu().numpy()) if profile else (d, e)


def shard_range(chi: int, rank: int, nranks: int):
    m0, m1 = c_int(0), c_int(0)
    if load_library().qrctm_shard_range(chi, rank, nranks, byref(m0), byref(m1)) != QRCTM_OK:
        raise QrctmError("qrctm_shard_range: invalid arguments")
    return m0.value, m1.value


def shard_exchange(Cn, Tn, rank: int, nranks: int, group=None):
    """The one exchange step of a sharded iteration (include/qrctm.h, NEXT-4), in place on every rank:
    Tn (chi rows of D^2 chi doubles; this rank's rows filled, zeros elsewhere) becomes the full T',
    Cn (partial) the full C'.  Equal slices: all-gather of the row blocks; ragged split: sum over ranks."""
    import torch.distributed as dist
    chi = Tn.shape[0]
    if chi % nranks == 0:
        mine = Tn.view(nranks, -1)[rank].clone()
        dist.all_gather_into_tensor(Tn.view(-1), mine, group=group)
    else:
        dist.all_reduce(Tn, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(Cn, op=dist.ReduceOp.SUM, group=group)


def eigh_top_f64(A, k: int):
    """(lam, U): the k eigenpairs of largest |lambda| of a symmetric torch CUDA float64 matrix through
    qrctm_eigh_top_f64 (A is copied; the library destroys its input)."""
    import torch
    lib = load_library()
    n = A.shape[0]
    nbytes = lib.qrctm_eigh_work_bytes(n, k)
    if nbytes == 0:
        raise QrctmError("qrctm_eigh_work_bytes: unsupported (n, k)")
    W = A.contiguous().clone()
    lam = torch.empty((k,), dtype=torch.float64, device="cuda")
    U = torch.empty((n, k), dtype=torch.float64, device="cuda")
    work = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    rc = lib.qrctm_eigh_top_f64(c_void_p(torch.cuda.current_stream().cuda_stream), n, k, _ptr(W), _ptr(lam), _ptr(U),
                                c_void_p(work.data_ptr()))
    if rc != QRCTM_OK:
        raise QrctmError(f"qrctm_eigh_top_f64 failed: {rc}")
    torch.cuda.current_stream().synchronize()
    return lam, U


def probe_fp64(kind: int, iters: int = 20000) -> float:
    lib = load_library()
    t = c_double(0.0)
    rc = lib.qrctm_probe_fp64(kind, iters, byref(t))
    if rc != QRCTM_OK:
        raise QrctmError(f"qrctm_probe_fp64 failed: {rc}")
    return t.value


def version() -> str:
    return load_library().qrctm_version().decode()
