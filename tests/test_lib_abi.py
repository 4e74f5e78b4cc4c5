"""CPU-only checks of the boundary: the library builds, loads without a GPU and
exports every symbol include/qrctm.h declares; invalid arguments are rejected;
the product path fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os
import re

import pytest

import paper_2505_00494_b200 as pkg
from paper_2505_00494_b200 import build as qbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    qbuild.build()
    return pkg.load_library()


def test_header_symbols_all_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "qrctm.h")).read()
    declared = set(re.findall(r"\b(qrctm_[A-Za-z0-9_]+)\s*\(", hdr))
    assert declared == set(pkg.SYMBOLS), declared ^ set(pkg.SYMBOLS)
    for s in declared:
        assert hasattr(lib, s), s


def test_links_no_vendor_math_library():
    out = os.popen(f"ldd {pkg.LIB_PATH}").read()
    for bad in ("cublas", "cusolver", "libtorch", "cudnn", "cutlass"):
        assert bad not in out.lower(), out
    assert "libcudart" in out


def test_invalid_arguments_rejected(lib):
    assert lib.qrctm_workspace_bytes(0, 2, 8) == 0
    assert lib.qrctm_workspace_bytes(2, 0, 8) == 0
    assert lib.qrctm_workspace_bytes(2, 2, 0) == 0
    n = lib.qrctm_workspace_bytes(2, 7, 196)
    m = 196 * 49
    assert 2 * 8 * m * m < n < 4 * 8 * m * m + (1 << 30)      # P, S (m^2 each) and the layered P1 (2 m^2) dominate
    h = ctypes.c_void_p()
    assert lib.qrctm_create(0, 2, 8, ctypes.byref(h)) == -1
    assert lib.qrctm_create(2, 2, 8, None) == -1
    assert lib.qrctm_destroy(None) == -1
    assert lib.qrctm_step(None) == -1
    assert lib.qrctm_qr_work_bytes(0, 1) == 0
    t = ctypes.c_double()
    assert lib.qrctm_probe_fp64(7, 10, ctypes.byref(t)) == -1
    assert b"qrctm" in lib.qrctm_version()
    # NEXT-2 / NEXT-4 entry points: argument checks need no device
    assert lib.qrctm_eigh_work_bytes(0, 1) == 0 and lib.qrctm_eigh_work_bytes(8, 9) == 0
    assert lib.qrctm_eigh_work_bytes(14001, 4) == 0 and lib.qrctm_eigh_work_bytes(9604, 196) > 8 * 4 * 9604 * 196
    assert lib.qrctm_eigh_top_f64(None, 4, 2, None, None, None, None) == -1
    for f in (lib.qrctm_init_bulk, lib.qrctm_shard_finish):
        assert f(None) == -1
    assert lib.qrctm_eig_step(None, 4) == -1 and lib.qrctm_warmup(None, 1) == -1
    assert lib.qrctm_shard_front(None, 0, 1) == -1
    m0, m1 = ctypes.c_int(), ctypes.c_int()
    assert lib.qrctm_shard_range(8, 0, 0, ctypes.byref(m0), ctypes.byref(m1)) == -1
    assert lib.qrctm_shard_range(8, 3, 3, ctypes.byref(m0), ctypes.byref(m1)) == -1
    assert lib.qrctm_shard_range(8, 1, 3, ctypes.byref(m0), ctypes.byref(m1)) == 0 and (m0.value, m1.value) == (3, 6)
    assert lib.qrctm_get_chi(None, None, None) == -1
    # stand-alone GEMM with a scratch buffer: null operands, bad path, misaligned / inconsistent scratch
    P = ctypes.c_void_p
    fake = P(256)
    assert lib.qrctm_gemm_f64_ws(None, 0, 1, 4, 4, 4, None, 4, None, 4, None, 4, None, 0) == -1
    assert lib.qrctm_gemm_f64_ws(None, 5, 1, 4, 4, 4, fake, 4, fake, 4, fake, 4, None, 0) == -1
    assert lib.qrctm_gemm_f64_ws(None, 0, 1, 4, 4, 4, fake, 4, fake, 4, fake, 4, P(8), 64) == -1
    assert lib.qrctm_gemm_f64_ws(None, 0, 1, 4, 4, 4, fake, 4, fake, 4, fake, 4, None, 64) == -1


def test_no_cpu_fallback_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = ctypes.c_void_p()
    assert lib.qrctm_create(2, 2, 8, ctypes.byref(h)) == -3       # QRCTM_ERR_CUDA
    assert not h.value
    with pytest.raises(pkg.QrctmError):
        pkg.QRCTM(2, 2, 8)


def test_product_path_does_not_import_oracle():
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2505_00494_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(root, f)).read()
                assert "oracle" not in src.replace("no oracle", ""), f
    src = open(os.path.join(ROOT, "qrctm_inputs", "__init__.py")).read()
    assert "import oracle" not in src and "from oracle" not in src
    osrc = open(os.path.join(ROOT, "oracle", "ctmrg.py")).read()
    assert "import paper_2505" not in osrc and "from paper_2505" not in osrc
