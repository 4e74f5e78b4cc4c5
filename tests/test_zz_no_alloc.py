"""The allocation-free GEMM entry (qrctm_gemm_f64_noalloc: K-splitting scratch in a static device array) against the
existing path (qrctm_gemm_f64_ws with a caller-provided scratch buffer) and NumPy, two calls in a row sharing the
scratch.  Collected last on purpose (the run uses pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import paper_2505_00494_b200 as pkg


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2505_00494_b200 import build as b
    b.build()


def rel(x, y):
    return np.linalg.norm(x - y) / np.linalg.norm(y)


def test_noalloc_gemm_matches_existing_path_two_calls_in_a_row():
    import torch
    g = np.random.default_rng(11)
    # call 1: C' = T'^T W of cfg4 (long K, small output: K is split); call 2: a different, smaller shape right after it,
    # so stale partials of call 1 would show; then call 1's inputs again (bitwise reproducible)
    shapes = [(196, 196, 9604), (100, 77, 2500), (196, 196, 9604)]
    outs = []
    for call, (M, N, K) in enumerate(shapes):
        gg = np.random.default_rng(M + N + K)
        A = gg.standard_normal((K, M)); B = gg.standard_normal((K, N))
        Ad, Bd = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
        out = torch.full((M, N), float("nan"), dtype=torch.float64, device="cuda")
        free0 = torch.cuda.mem_get_info()[0]
        pkg.gemm_f64_noalloc(Ad, Bd, out, transA=True)
        torch.cuda.synchronize()
        if call == 2:          # same kernels as call 0 (nothing left to load lazily): the call took no device memory
            assert torch.cuda.mem_get_info()[0] == free0
        ref = pkg.gemm_f64(Ad, Bd, transA=True, work_bytes=64 << 20).cpu().numpy()
        o = out.cpu().numpy()
        assert rel(o, ref) < 1e-13 and rel(o, A.T @ B) < 1e-13
        outs.append(o)
    assert np.array_equal(outs[0], outs[2])


def test_noalloc_gemm_plain_layout_and_size_limit():
    import torch
    g = np.random.default_rng(5)
    A = g.standard_normal((64, 300)); B = g.standard_normal((300, 33))          # transA = 0
    out = torch.empty((64, 33), dtype=torch.float64, device="cuda")
    pkg.gemm_f64_noalloc(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), out)
    assert rel(out.cpu().numpy(), A @ B) < 1e-13
    big = torch.zeros((8, 300), dtype=torch.float64, device="cuda")
    with pytest.raises(pkg.QrctmError, match="65536"):
        pkg.gemm_f64_noalloc(big, torch.zeros((8, 257), dtype=torch.float64, device="cuda"),
                             torch.empty((300, 257), dtype=torch.float64, device="cuda"), transA=True)
