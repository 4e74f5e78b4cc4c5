"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are the north_star's:
single step <= 1e-11 relative Frobenius on C and T (after the R-sign gauge fix),
converged run <= 1e-9 on kappa and the top-10 corner spectrum.  Sub-steps
(SURVEY.md P12): 1e-13 per GEMM, Q within cond(c~) * 1e-14."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import paper_2505_00494_b200 as pkg
from oracle import ctmrg as o
from qrctm_inputs import CONFIGS, gen_config, random_isometry


def rel(x, y):
    x = np.asarray(x); y = np.asarray(y)
    return np.linalg.norm(x - y) / np.linalg.norm(y)


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2505_00494_b200 import build as b
    b.build()


def torch_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


# ------------------------------------------------------------------ sub-steps
@pytest.mark.parametrize("M,N,K,transA", [
    (8, 32, 8, False), (32, 32, 8, True), (196, 9604, 196, False), (324, 324, 36, True),
    (1000, 333, 77, True), (129, 257, 65, True), (64, 64, 2401, True), (37, 41, 1000, True),
    (300, 300, 3, False), (1, 1, 1, True), (5, 7, 1, False), (2500, 100, 2500, True),
])
@pytest.mark.parametrize("path", [0, 1])
def test_gemm_f64_matches_numpy(M, N, K, transA, path):
    g = np.random.default_rng(M * 7 + N * 3 + K)
    A = g.standard_normal((K, M) if transA else (M, K))
    B = g.standard_normal((K, N))
    ref = (A.T if transA else A) @ B
    out = pkg.gemm_f64(torch_dev(A), torch_dev(B), transA=transA, path=path).cpu().numpy()
    assert rel(out, ref) < 1e-13


def test_gemm_odd_leading_dimension_views():
    import torch
    g = np.random.default_rng(0)
    A = torch_dev(g.standard_normal((70, 131)))[:, :129]       # lda = 131 (odd) -> scalar loads
    B = torch_dev(g.standard_normal((70, 59)))[:, 1:58]        # misaligned base
    out = pkg.gemm_f64(A, B, transA=True).cpu().numpy()
    assert rel(out, A.cpu().numpy().T @ B.cpu().numpy()) < 1e-13


_QR_SHAPES = [(32, 8), (324, 36), (1024, 64), (50, 50), (7, 1), (333, 17), (16, 16),
              (2500, 100), (40, 33), (9604, 196), (3000, 150), (112, 112), (5000, 64), (1792, 112), (4096, 50),
              (15000, 24), (40000, 40),   # 16-CTA cluster; global-memory panel path
              (5120, 130), (5121, 130), (2000, 113),   # one-launch trailing update: its row limit, one past it, ragged slab
              (10241, 40), (12289, 48), (16400, 33), (20480, 20), (20481, 20)]   # tall register panels: 48 / 64 / 80 rows
                                                                                  # per thread, and one row past them
_QR_SHAPES += [(208, 208), (5000, 207), (3000, 208), (3000, 209), (4000, 177)]   # CholeskyQR2's column limit (208) +- 1, odd n
# paths: 0 automatic (CholeskyQR2 for 48 <= n <= 208, Householder when its device-side check fails or outside that
# range), 1 per-reflector (level-2; only on small cases), 2 blocked Householder, 3 Householder automatic,
# 4 CholeskyQR2 whenever n <= 208
_QR_CASES = [(r, c, p) for p in (0, 1, 2, 3, 4) for (r, c) in _QR_SHAPES if not (p == 1 and r * c > 200000)]


@pytest.mark.parametrize("rows,cols,path", _QR_CASES)
def test_qr_f64_matches_oracle(rows, cols, path):
    g = np.random.default_rng(rows + cols)
    X = g.standard_normal((rows, cols))
    Q, R = pkg.qr_f64(torch_dev(X), path=path)
    Q, R = Q.cpu().numpy(), R.cpu().numpy()
    Qo, Ro = o.qr_pos(X)
    cond = np.linalg.cond(X)
    assert np.all(np.tril(R, -1) == 0.0) and np.all(np.diag(R) >= 0.0)
    assert np.linalg.norm(Q.T @ Q - np.eye(cols)) < cols * 2e-15
    assert rel(Q @ R, X) < 1e-14
    assert rel(R, Ro) < 1e-14 * max(cond, 10)
    assert rel(Q, Qo) < 1e-14 * max(cond, 10)


@pytest.mark.parametrize("n", [1, 2, 7, 16, 17, 36, 100, 150, 196, 207, 208])
def test_chol_inv_kernel_against_lapack(n):
    """The n x n factorisation inside CholeskyQR2 (qrctm_chol_inv_f64): R = chol(G)^T, R^-1, ||G - I||_F, breakdown flag."""
    g = np.random.default_rng(n)
    X = g.standard_normal((3 * n + 5, n))
    G = X.T @ X / (3 * n)
    R, Ri, st, dev = pkg.chol_inv_f64(torch_dev(G))
    R, Ri = R.cpu().numpy(), Ri.cpu().numpy()
    Rn = np.linalg.cholesky(G).T
    cond = np.linalg.cond(Rn)
    assert st == 0 and abs(dev - np.linalg.norm(G - np.eye(n))) < 1e-12 * max(1.0, dev)
    assert np.all(np.tril(R, -1) == 0.0) and np.all(np.tril(Ri, -1) == 0.0) and np.all(np.diag(R) > 0)
    assert rel(R, Rn) < 1e-14 * max(cond, 10)
    assert np.linalg.norm(Ri @ Rn - np.eye(n)) < 1e-14 * n * max(cond, 10)
    G[n // 2, n // 2] = -1.0                                # not positive definite: breakdown must be flagged
    assert pkg.chol_inv_f64(torch_dev(G))[2] == 1


def test_qr_maximum_column_count():
    """The build's limit chi <= 800 (form-Q back substitution keeps chi/16 blocks in shared memory): 800 columns work
    (blocked Householder path, 50 panels), 801 are rejected with QRCTM_ERR_INVALID_ARG instead of failing at launch."""
    g = np.random.default_rng(800)
    X = g.standard_normal((1000, 800))
    Q, R = pkg.qr_f64(torch_dev(X), path=0)
    Q, R = Q.cpu().numpy(), R.cpu().numpy()
    assert np.linalg.norm(Q.T @ Q - np.eye(800)) < 800 * 2e-15 and rel(Q @ R, X) < 1e-13
    assert np.all(np.diag(R) >= 0) and np.all(np.tril(R, -1) == 0)
    with pytest.raises(pkg.QrctmError):
        pkg.qr_f64(torch_dev(g.standard_normal((900, 801))), path=0)
    assert pkg.load_library().qrctm_workspace_bytes(2, 1, 801) == 0 and pkg.load_library().qrctm_workspace_bytes(2, 1, 800) > 0


def test_qr_rank_deficient_is_still_valid():
    g = np.random.default_rng(3)
    X = g.standard_normal((200, 6)) @ g.standard_normal((6, 12))       # rank 6 < 12 (hazard H1)
    for path in (0, 1, 2, 3, 4):
        Q, R = pkg.qr_f64(torch_dev(X), path=path)
        Q, R = Q.cpu().numpy(), R.cpu().numpy()
        assert np.linalg.norm(Q.T @ Q - np.eye(12)) < 1e-13
        assert rel(Q @ R, X) < 1e-13 and np.all(np.diag(R) >= 0.0)
    Q, R = pkg.qr_f64(torch_dev(X))
    Q, R = Q.cpu().numpy(), R.cpu().numpy()
    assert np.linalg.norm(Q.T @ Q - np.eye(12)) < 1e-13
    assert rel(Q @ R, X) < 1e-13 and np.all(np.diag(R) >= 0.0)


@pytest.mark.parametrize("expo", [1, 3, 5, 7, 9, 12])
def test_qr_graded_conditioning_automatic_path(expo):
    """The automatic path over a range of cond(X) = 10^expo: CholeskyQR2 where its device-side check
    (||Q1^T Q1 - I||_F <= 1e-4, no pivot breakdown) passes, Householder beyond -- always orthonormal to rounding,
    residual at rounding level, and Q, R within cond x 1e-14 of the oracle (until cond eps ~ 1)."""
    g = np.random.default_rng(expo)
    U, _ = np.linalg.qr(g.standard_normal((3000, 100)))
    V, _ = np.linalg.qr(g.standard_normal((100, 100)))
    X = np.ascontiguousarray((U * np.logspace(0, -expo, 100)) @ V.T)
    Q, R = pkg.qr_f64(torch_dev(X), path=0)
    Q, R = Q.cpu().numpy(), R.cpu().numpy()
    assert np.all(np.tril(R, -1) == 0.0) and np.all(np.diag(R) >= 0.0)
    assert np.linalg.norm(Q.T @ Q - np.eye(100)) < 100 * 2e-15
    assert rel(Q @ R, X) < 1e-14
    Qo, Ro = o.qr_pos(X)
    assert rel(R, Ro) < 1e-14 * 10.0 ** expo
    if expo <= 9:
        assert rel(Q, Qo) < 1e-14 * 10.0 ** expo * 10


def test_step_with_rank_deficient_corner_takes_the_householder_fallback_inside_the_graph():
    """A product-state A makes c~ numerically rank-deficient (hazard H1): CholeskyQR2's device-side check fails and the
    captured step runs the Householder body of its conditional node.  Graph replay, direct launches and the forced
    Householder path must agree on the gauge-invariant results (kappa exact for a product state, pin P6)."""
    d, D, chi = 2, 3, 12
    g = np.random.default_rng(5)
    phi, v = g.standard_normal(d), g.standard_normal(D)
    A = np.einsum("s,u,l,d,r->suldr", phi, v, v, v, v).copy()
    _, C0, T0 = gen_config(d, D, chi, 7)
    ks = []
    for qr_path, graph in ((4, 1), (4, 0), (3, 1)):
        h = pkg.QRCTM(d, D, chi)
        h.set_option(pkg.OPT_QR_PATH, qr_path)
        h.set_option(pkg.OPT_USE_GRAPH, graph)
        h.set_A(A); h.set_env(C0, T0)
        h.run(25, -1.0)
        Q, R = h.get_qr()
        assert np.linalg.norm(Q.T @ Q - np.eye(chi)) < 1e-13
        ks.append(h.norm_per_site())
        h.close()
    exact = (phi @ phi) * (v @ v) ** 4
    for k in ks:
        assert abs(k / exact - 1) < 1e-11


@pytest.mark.parametrize("d,D,chi,seed", [(2, 2, 8, 0), (2, 3, 36, 1), (3, 2, 5, 4), (2, 3, 7, 5), (1, 1, 4, 2)])
def test_build_a_bit_exact_layout(d, D, chi, seed):
    A, C0, T0 = gen_config(d, D, chi, seed)
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A)
    a = h.get_a()
    assert rel(a, o.build_a(A)) < 1e-15 if np.linalg.norm(a) > 0 else True
    h.close()


# ------------------------------------------------------------------ single step
def _one_step(d, D, chi, seed, corner_mode=0, path=0, absorb=0):
    A, C0, T0 = gen_config(d, D, chi, seed)
    h = pkg.QRCTM(d, D, chi)
    h.set_option(pkg.OPT_CORNER_MODE, corner_mode)
    h.set_option(pkg.OPT_GEMM_PATH, path)
    h.set_option(pkg.OPT_ABSORB_MODE, absorb)
    h.set_A(A)
    h.set_env(C0, T0)
    C_in, T_in = h.get_env()
    h.step()
    out = dict(C=h.get_env()[0], T=h.get_env()[1], QR=h.get_qr(), raw=h.get_raw(), Cin=C_in, Tin=T_in,
               ratio=h.r_diag_ratio(), launches=h.launch_count())
    h.close()
    a = o.build_a(A)
    Cr, Tr = o.normalize(C0, T0)
    s = o.qr_step(Cr, Tr, a, corner="accelerated" if corner_mode == 0 else "enlarged")
    Co, To = o.normalize(s["Cn"], s["Tn"])
    return out, s, (Cr, Tr, Co, To)


STEP_CASES = [(2, 2, 8, 0), (2, 3, 36, 1), (2, 4, 64, 2), (3, 2, 5, 7), (2, 3, 7, 8), (2, 1, 3, 9), (2, 2, 1, 3)]


@pytest.mark.parametrize("d,D,chi,seed", STEP_CASES)
def test_single_step_parity(d, D, chi, seed):
    out, s, (Cr, Tr, Co, To) = _one_step(d, D, chi, seed)
    assert rel(out["Cin"], Cr) < 1e-14 and rel(out["Tin"], Tr) < 1e-14
    Q, R = out["QR"]
    cond = np.linalg.cond(s["X"])
    assert rel(R, s["R"]) < 1e-14 * max(cond, 10)
    assert rel(Q, s["Q"]) < 1e-14 * max(cond, 10)
    assert np.all(np.diag(R) >= 0) and np.all(np.tril(R, -1) == 0)
    Cn, Tn = out["raw"]
    assert rel(Tn, s["Tn"]) < 1e-11 and rel(Cn, s["Cn"]) < 1e-11
    assert rel(out["C"], Co) < 1e-11
    assert rel(out["T"], To) < 1e-11
    assert abs(np.linalg.norm(out["C"]) - 1) < 1e-14 and abs(np.linalg.norm(out["T"]) - 1) < 1e-14
    assert np.array_equal(out["C"], out["C"].T)
    assert np.array_equal(out["T"], out["T"].transpose(2, 1, 0))
    d_ = np.diag(s["R"])
    assert abs(out["ratio"] - d_.min() / d_.max()) < 1e-10


@pytest.mark.parametrize("d,D,chi,seed", [(2, 2, 8, 0), (2, 3, 12, 1), (2, 3, 7, 8),
                                          (2, 4, 64, 2), (2, 5, 100, 3), (2, 7, 196, 4)])   # ... cfg2, cfg3a, cfg4
def test_single_step_enlarged_corner_mode(d, D, chi, seed):
    """K6': the enlarged corner C~ (E5) and C' = Q^T C~ Q (E4'), "the standard diagram on the left-hand side" of
    Fig. 1(f), up to BASELINE.json's full sizes (cfg4: C~ is 9604 x 9604), against the oracle's
    enlarged-corner branch and against the accelerated update (E4)."""
    out, s, (Cr, Tr, Co, To) = _one_step(d, D, chi, seed, corner_mode=1)
    assert rel(out["raw"][0], s["Cn"]) < 1e-11 and rel(out["raw"][1], s["Tn"]) < 1e-11
    assert rel(out["C"], Co) < 1e-11 and rel(out["T"], To) < 1e-11
    acc, _, _ = _one_step(d, D, chi, seed, corner_mode=0)
    assert rel(out["raw"][0], acc["raw"][0]) < 1e-12            # Fig. 1(f): (E4) == (E4')


def test_single_step_reference_gemm_path_agrees():
    out0, s, _ = _one_step(2, 3, 20, 1, path=0)
    out1, _, _ = _one_step(2, 3, 20, 1, path=1)
    assert rel(out0["T"], out1["T"]) < 1e-12 and rel(out0["C"], out1["C"]) < 1e-12


def test_step_is_deterministic_bitwise():
    a, _, _ = _one_step(2, 3, 36, 1)
    b, _, _ = _one_step(2, 3, 36, 1)
    assert np.array_equal(a["C"], b["C"]) and np.array_equal(a["T"], b["T"])


@pytest.mark.parametrize("d,D,chi,ncols,seed", [(2, 2, 6, 6, 3), (2, 3, 36, 36, 1), (2, 3, 20, 14, 2), (3, 2, 9, 5, 4),
                                                (2, 4, 64, 64, 5), (2, 5, 100, 100, 6)])
def test_edge_update_with_arbitrary_isometry(d, D, chi, ncols, seed):
    """K3-K5 alone (qrctm_edge_update) with a seeded random isometry that is NOT a QR factor of c~,
    square and with fewer columns than chi, against the oracle's (E3)."""
    A, C0, T0 = gen_config(d, D, chi, seed)
    U = random_isometry(chi * D * D, ncols, seed + 50)
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A); h.set_env(C0, T0)
    C, T = o.normalize(C0, T0)
    Tn = h.edge_update(U)
    assert Tn.shape == (ncols, D * D, ncols)
    assert rel(Tn, o.edge_update(U, T, o.build_a(A))) < 1e-13
    Tn2 = h.edge_update(torch_dev(U), device=True).cpu().numpy()          # device pointers
    assert np.array_equal(Tn, Tn2)
    C1, T1 = h.get_env()
    assert rel(C1, C) < 1e-14 and rel(T1, T) < 1e-14                      # environment untouched
    h.close()


def test_gpu_step_edge_is_the_oracle_contraction_of_its_own_q():
    d, D, chi = 2, 2, 6
    A, C0, T0 = gen_config(d, D, chi, 3)
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A); h.set_env(C0, T0); h.step()
    Q, R = h.get_qr()
    _, Tn = h.get_raw()
    C, T = o.normalize(C0, T0)
    assert rel(Tn, o.edge_update(Q, T, o.build_a(A))) < 1e-13
    h.close()


# ------------------------------------------------------------------ runs
def _oracle_steps(A, C0, T0, n):
    a = o.build_a(A)
    C, T = o.normalize(C0, T0)
    for _ in range(n):
        s = o.qr_step(C, T, a)
        C, T = o.normalize(s["Cn"], s["Tn"])
    return C, T, a


def test_cfg0_converged_run_parity():
    c = CONFIGS["cfg0"]
    A, C0, T0 = gen_config(c["d"], c["D"], c["chi"], c["seed"])
    h = pkg.QRCTM(c["d"], c["D"], c["chi"])
    h.set_A(A); h.set_env(C0, T0)
    it, dl = h.run(500, 1e-12)
    a = o.build_a(A)
    Co, To, ito, dlo, _ = o.run(C0, T0, a, "qr", 500, 1e-12)
    assert abs(it - ito) <= 1 and dl < 1e-12
    k, ko = h.norm_per_site(), o.kappa(Co, To, a)
    assert abs(k / ko - 1) < 1e-9
    s, so = h.get_corner_spectrum(), o.spectrum(Co)
    assert np.max(np.abs(s[:8] - so[:8]) / so[:8]) < 1e-9
    assert abs(np.sum(s ** 2) - 1) < 1e-13 and np.all(np.diff(s) <= 0)
    if it == ito:
        C, T = h.get_env()
        assert rel(C, Co) < 1e-9 and rel(T, To) < 1e-9
    h.close()


def test_cfg0_fifty_iterations_fixed_count():
    c = CONFIGS["cfg0"]
    A, C0, T0 = gen_config(c["d"], c["D"], c["chi"], c["seed"])
    h = pkg.QRCTM(c["d"], c["D"], c["chi"])
    h.set_A(A); h.set_env(C0, T0)
    it, dl = h.run(50, 1e-12)
    assert it == 50
    Co, To, a = _oracle_steps(A, C0, T0, 50)
    C, T = h.get_env()
    assert rel(C, Co) < 1e-10 and rel(T, To) < 1e-10
    assert np.max(np.abs(h.get_corner_spectrum() - o.spectrum(Co))) < 1e-12
    h.close()


def test_cfg1_fixed_count_and_kappa():
    c = CONFIGS["cfg1"]
    A, C0, T0 = gen_config(c["d"], c["D"], c["chi"], c["seed"])
    h = pkg.QRCTM(c["d"], c["D"], c["chi"])
    h.set_A(A); h.set_env(C0, T0)
    for _ in range(20):
        h.step()
    Co, To, a = _oracle_steps(A, C0, T0, 20)
    C, T = h.get_env()
    assert rel(C, Co) < 1e-9 and rel(T, To) < 1e-9
    s, so = h.get_corner_spectrum(), o.spectrum(Co)
    assert np.max(np.abs(s[:10] - so[:10]) / so[:10]) < 1e-9
    assert abs(h.norm_per_site() / o.kappa(Co, To, a) - 1) < 1e-9
    h.close()


def test_spectrum_kernel_against_lapack():
    import torch
    # chi <= 24: one fused kernel (one-warp tridiagonalisation); <= 64 / 128: the register-resident kernels (256 / 512
    # threads); <= 216 / 236: shared-memory tridiagonalisations; above: the multi-CTA tridiagonalisation of the eigen step
    for chi, seed in [(1, 0), (2, 1), (3, 10), (8, 2), (24, 11), (25, 12), (31, 17), (32, 13), (33, 14), (36, 3), (40, 15),
                      (41, 16), (63, 18), (64, 19), (65, 20), (100, 4), (127, 21), (128, 22), (129, 23), (196, 5), (236, 6), (237, 7),
                      (400, 8), (700, 9)]:
        A, C0, T0 = gen_config(2, 1, chi, seed)
        h = pkg.QRCTM(2, 1, chi)
        h.set_A(A); h.set_env(C0, T0)
        C, _ = h.get_env()
        s = h.get_corner_spectrum()
        assert np.max(np.abs(s - o.spectrum(C))) < 5e-15 * chi, chi
        h.close()


@pytest.mark.parametrize("n", [1, 2, 3, 8, 31, 32, 33, 64, 65, 100, 161, 196, 216])
def test_tridiag_kernel_preserves_the_spectrum(n):
    """qrctm_tridiag_f64 (K8's first stage): the tridiagonal (d, e) it returns is orthogonally similar to C, so the
    eigenvalues agree with LAPACK's to rounding; also on a rank-one matrix (the trailing block is rounding noise)."""
    g = np.random.default_rng(n)
    C = g.standard_normal((n, n)); C = C + C.T; C /= np.linalg.norm(C)
    for M in (C, np.ones((n, n)) / n):
        d, e = pkg.tridiag_f64(torch_dev(M))
        d, e = d.cpu().numpy(), e.cpu().numpy()
        T = np.diag(d) + np.diag(e[1:], 1) + np.diag(e[1:], -1)
        assert e[0] == 0.0
        assert np.max(np.abs(np.linalg.eigvalsh(T) - np.linalg.eigvalsh(M))) < 5e-15 * max(n, 4)


@pytest.mark.parametrize("name,n", [("identity", 30), ("diag", 37), ("block", 32), ("ones", 33), ("rank2", 40), ("zero_tail", 20),
                                    ("identity", 64), ("block", 56), ("ones", 16), ("rank2", 61), ("zero_tail", 50), ("diag", 12),
                                    ("identity", 100), ("block", 128), ("ones", 90), ("rank2", 113), ("zero_tail", 70), ("diag", 77)])
def test_spectrum_small_structured_matrices(name, n):
    """The small tridiagonalisations (one warp for n <= 24, registers for n <= 64) on matrices whose reflectors vanish or
    whose trailing block is rounding noise (n <= 128: 512-thread register kernel): identity, diagonal, block-diagonal of all-ones blocks, all ones, rank two, a
    matrix with an exactly zero tail."""
    g = np.random.default_rng(n)
    if name == "identity": C = np.eye(n)
    elif name == "diag": C = np.diag(np.arange(1.0, n + 1))
    elif name == "block": C = np.kron(np.eye(n // 8), np.ones((8, 8)))
    elif name == "ones": C = np.ones((n, n))
    elif name == "rank2":
        v, w = g.standard_normal(n), g.standard_normal(n)
        C = np.outer(v, v) - 0.5 * np.outer(w, w)
    else:
        C = np.zeros((n, n)); B = g.standard_normal((5, 5)); C[:5, :5] = B + B.T
    A, C0, T0 = gen_config(2, 1, n, 1)
    h = pkg.QRCTM(2, 1, n)
    h.set_A(A); h.set_env(C, T0)
    Cn, _ = h.get_env()
    s = h.get_corner_spectrum()
    assert np.max(np.abs(s - o.spectrum(Cn))) < 5e-15 * n
    h.close()


def test_k8_paths_agree():
    A, C0, T0 = gen_config(2, 1, 150, 3)
    out = []
    for path in (0, 1):
        h = pkg.QRCTM(2, 1, 150)
        h.set_option(pkg.OPT_K8_PATH, path)
        h.set_A(A); h.set_env(C0, T0)
        out.append(h.get_corner_spectrum())
        h.close()
    assert np.max(np.abs(out[0] - out[1])) < 1e-14


def test_errors_and_not_ready():
    h = pkg.QRCTM(2, 2, 4)
    with pytest.raises(pkg.QrctmError):
        h.step()
    A, C0, T0 = gen_config(2, 2, 4, 0)
    h.set_A(A)
    with pytest.raises(pkg.QrctmError):
        h.run(3, 1e-3)
    with pytest.raises(pkg.QrctmError):
        h.set_env(np.zeros((4, 4)), T0)            # zero Frobenius norm -> NUMERIC
    with pytest.raises(pkg.QrctmError):
        h.set_option(99, 0)
    h.close()


def test_device_pointers_accepted_and_set_A_keeps_env():
    import torch
    A, C0, T0 = gen_config(2, 2, 8, 0)
    h = pkg.QRCTM(2, 2, 8)
    h.set_A(torch_dev(A)); h.set_env(torch_dev(C0), torch_dev(T0))
    h.step()
    C1, T1 = h.get_env(device=True)
    h.set_A(A * 0.5)                                # environment is kept
    C2, T2 = h.get_env()
    assert np.array_equal(C1.cpu().numpy(), C2) and np.array_equal(T1.cpu().numpy(), T2)
    h.close()


def test_ising_onsager_on_gpu():
    from tests.brute import ising_A, onsager_ln_kappa
    K = 0.3
    A = ising_A(K)
    _, C0, T0 = gen_config(2, 2, 16, 1)
    h = pkg.QRCTM(2, 2, 16)
    h.set_A(A); h.set_env(C0, T0)
    h.run(300, 1e-13)
    assert abs(np.log(h.norm_per_site()) - onsager_ln_kappa(K)) < 1e-10
    h.close()


def test_overlapped_check_is_bitwise_identical_to_serial():
    """qrctm_run with the convergence check overlapped on the side stream must give the same
    iteration count, delta and environment as the strictly serial driver."""
    A, C0, T0 = gen_config(2, 3, 24, 0)
    res = []
    for overlap in (1, 0):
        h = pkg.QRCTM(2, 3, 24)
        h.set_option(pkg.OPT_OVERLAP_CHECK, overlap)
        h.set_A(A); h.set_env(C0, T0)
        it, dl = h.run(400, 1e-9)
        C, T = h.get_env()
        it2, dl2 = h.run(7, -1.0)                  # fixed count afterwards
        C2, T2 = h.get_env()
        res.append((it, dl, C, T, it2, dl2, C2, T2, h.get_corner_spectrum()))
        h.close()
    a, b = res
    assert a[0] == b[0] and a[1] == b[1] and a[4] == b[4] == 7 and a[5] == b[5]
    assert a[0] < 400
    for i in (2, 3, 6, 7, 8):
        assert np.array_equal(a[i], b[i])


def test_history_ring_buffer_matches_oracle_run():
    """qrctm_get_history: per-iteration delta, ||C'||_F, ||T'||_F, min/max R_kk against the oracle's run history."""
    A, C0, T0 = gen_config(2, 3, 20, 1)
    a = o.build_a(A)
    h = pkg.QRCTM(2, 3, 20)
    h.set_A(A); h.set_env(C0, T0)
    it, dl = h.run(12, -1.0)
    rec, n = h.get_history()
    assert n == 12 and rec.shape == (12, 4)
    C, T = o.normalize(C0, T0)
    s_prev = o.spectrum(C)
    for k in range(12):
        st = o.qr_step(C, T, a)
        d = np.diag(st["R"])
        assert abs(rec[k, 1] / np.linalg.norm(0.5 * (st["Cn"] + st["Cn"].T)) - 1) < 1e-9
        assert abs(rec[k, 2] / np.linalg.norm(0.5 * (st["Tn"] + st["Tn"].transpose(2, 1, 0))) - 1) < 1e-9
        assert abs(rec[k, 3] - d.min() / d.max()) < 1e-9
        C, T = o.normalize(st["Cn"], st["Tn"])
        s = o.spectrum(C)
        assert abs(rec[k, 0] - np.max(np.abs(s - s_prev))) < 1e-11
        s_prev = s
    assert rec[-1, 0] == dl
    h.set_option(pkg.OPT_CHECK_EVERY, 4)
    h.run(8, -1.0)
    rec, n = h.get_history(6)
    assert n == 20 and rec.shape == (6, 4)
    assert np.isnan(rec[0, 0]) and np.isfinite(rec[1, 0]) and np.isnan(rec[2, 0]) and np.isfinite(rec[5, 0])
    h.set_env(C0, T0)
    assert h.get_history()[1] == 0
    h.close()


def test_check_every_option():
    A, C0, T0 = gen_config(2, 2, 8, 0)
    h = pkg.QRCTM(2, 2, 8)
    h.set_option(pkg.OPT_CHECK_EVERY, 5)
    h.set_A(A); h.set_env(C0, T0)
    it, dl = h.run(500, 1e-12)
    assert it % 5 == 0 and it < 500
    Co, To, a = _oracle_steps(A, C0, T0, it)
    C, T = h.get_env()
    assert rel(C, Co) < 1e-9 and rel(T, To) < 1e-9
    h.close()


@pytest.mark.parametrize("name", ["cfg3a", "cfg3b", "cfg4"])
def test_full_size_single_step_parity(name):
    """North-star bar at BASELINE.json's full sizes, in the launch configuration bench.py times:
    relative Frobenius error <= 1e-11 on C and T after one step (after the R-sign gauge fix)."""
    c = CONFIGS[name]
    out, s, (Cr, Tr, Co, To) = _one_step(c["d"], c["D"], c["chi"], c["seed"])
    Q, R = out["QR"]
    cond = np.linalg.cond(s["X"])
    assert rel(R, s["R"]) < 1e-14 * max(cond, 10) and rel(Q, s["Q"]) < 1e-14 * max(cond, 10)
    assert np.linalg.norm(Q.T @ Q - np.eye(c["chi"])) < c["chi"] * 2e-15
    Cn, Tn = out["raw"]
    assert rel(Tn, s["Tn"]) < 1e-11 and rel(Cn, s["Cn"]) < 1e-11
    assert rel(out["C"], Co) < 1e-11 and rel(out["T"], To) < 1e-11
    assert np.array_equal(out["C"], out["C"].T) and np.array_equal(out["T"], out["T"].transpose(2, 1, 0))


def test_cfg3a_ten_steps_and_kappa_parity():
    c = CONFIGS["cfg3a"]
    A, C0, T0 = gen_config(c["d"], c["D"], c["chi"], c["seed"])
    h = pkg.QRCTM(c["d"], c["D"], c["chi"])
    h.set_A(A); h.set_env(C0, T0)
    it, dl = h.run(10, -1.0)
    assert it == 10
    Co, To, a = _oracle_steps(A, C0, T0, 10)
    C, T = h.get_env()
    assert rel(C, Co) < 1e-9 and rel(T, To) < 1e-9
    s, so = h.get_corner_spectrum(), o.spectrum(Co)
    assert np.max(np.abs(s[:10] - so[:10]) / so[:10]) < 1e-9
    assert abs(h.norm_per_site() / o.kappa(Co, To, a) - 1) < 1e-9
    h.close()


_LAYERED_SIZES = [(2, 2, 8, 0), (2, 3, 36, 1), (3, 2, 6, 7), (2, 4, 64, 2), (2, 5, 100, 3), (2, 7, 196, 4), (2, 3, 7, 8)]
# the reference GEMM (path 1) is only run on the small cases
_LAYERED_CASES = [sz + (p,) for p in (0, 1) for sz in _LAYERED_SIZES if not (p == 1 and sz[2] > 40)]


@pytest.mark.parametrize("d,D,chi,seed,path", _LAYERED_CASES)
def test_layered_absorption_matches_oracle_and_explicit(d, D, chi, seed, path):
    """NEXT-1: absorbing the ket and bra layers of A one after the other gives the same T' (and C')
    as the explicit double-layer tensor; odd chi silently uses the explicit path."""
    lay, s, (Cr, Tr, Co, To) = _one_step(d, D, chi, seed, absorb=1, path=path)
    assert rel(lay["raw"][1], s["Tn"]) < 1e-11 and rel(lay["raw"][0], s["Cn"]) < 1e-11
    assert rel(lay["C"], Co) < 1e-11 and rel(lay["T"], To) < 1e-11
    exp, _, _ = _one_step(d, D, chi, seed, absorb=0, path=path)
    assert rel(lay["raw"][1], exp["raw"][1]) < 1e-12


@pytest.mark.parametrize("d,D,chi,seed", [(2, 2, 8, 0), (3, 2, 5, 7), (2, 3, 7, 8), (2, 2, 20, 4), (2, 1, 3, 9)])
def test_small_whole_iteration_kernels_match_the_general_path(d, D, chi, seed):
    """Tiny problems run K1..K6 as one kernel, K7 as one and K8 as one (QRCTM_OPT_SMALL_PATH = 2; the default takes
    this path for chi <= 8): same step as the general multi-kernel path to rounding, same iteration count and delta
    history, far fewer launches."""
    A, C0, T0 = gen_config(d, D, chi, seed)
    out = {}
    for off in (0, 1):
        h = pkg.QRCTM(d, D, chi)
        h.set_option(pkg.OPT_SMALL_PATH, 1 if off else 2)
        h.set_A(A); h.set_env(C0, T0)
        h.step()
        Q, R = h.get_qr()
        raw = h.get_raw()
        n0 = h.launch_count()
        it, dl = h.run(12, -1.0)
        out[off] = (Q, R, raw, h.get_env(), h.get_corner_spectrum(), dl, h.launch_count() - n0, h.get_history()[0])
        h.close()
    s, g = out[0], out[1]
    cond = np.linalg.cond(g[1])
    assert rel(s[0], g[0]) < 1e-14 * max(cond, 10) and rel(s[1], g[1]) < 1e-14 * max(cond, 10)
    assert rel(s[2][0], g[2][0]) < 1e-12 and rel(s[2][1], g[2][1]) < 1e-12
    assert rel(s[3][0], g[3][0]) < 1e-10 and rel(s[3][1], g[3][1]) < 1e-10
    assert np.max(np.abs(s[4] - g[4])) < 1e-11 and abs(s[5] - g[5]) < 1e-10
    assert np.allclose(s[7][:, 1:], g[7][:, 1:], rtol=1e-9) and s[6] * 3 < g[6]


def test_small_path_default_is_by_measured_crossover():
    """QRCTM_OPT_SMALL_PATH = 0: the one-kernel path up to chi = 8, the general path above (where it is faster)."""
    for chi, small in ((8, True), (16, False)):
        A, C0, T0 = gen_config(2, 2, chi, 1)
        h = pkg.QRCTM(2, 2, chi)
        h.set_A(A); h.set_env(C0, T0)
        h.run(3, -1.0)
        n0 = h.launch_count()
        h.run(10, -1.0)
        per_step = (h.launch_count() - n0) / 10
        h.close()
        assert (per_step <= 3.5) == small, (chi, per_step)


@pytest.mark.parametrize("check_every", [2, 3, 7])
def test_device_side_run_loop_for_tiny_problems(check_every):
    """Tiny problems with CHECK_EVERY >= 2: qrctm_run is ONE kernel launch, the convergence decision is taken on the
    device.  Iteration count, delta, environment, history against the oracle's run with the same check interval, and
    against the pipelined host driver (QRCTM_OPT_SMALL_PATH = 1)."""
    c = CONFIGS["cfg0"]
    A, C0, T0 = gen_config(c["d"], c["D"], c["chi"], c["seed"])
    a = o.build_a(A)
    res = []
    for off in (0, 1):
        h = pkg.QRCTM(c["d"], c["D"], c["chi"])
        h.set_option(pkg.OPT_SMALL_PATH, off)
        h.set_option(pkg.OPT_CHECK_EVERY, check_every)
        h.set_A(A); h.set_env(C0, T0)
        n0 = h.launch_count()
        it, dl = h.run(400, 1e-11)
        res.append((it, dl, h.get_env(), h.launch_count() - n0, h.get_history()[1]))
        it2, dl2 = h.run(0, 1e-11)
        assert it2 == 0
        h.close()
    (it, dl, (C, T), nl, nh), (itg, dlg, (Cg, Tg), nlg, _) = res
    assert nl == 1 and nlg > 50 and nh == it
    assert it == itg and it % check_every == 0 and it < 400 and dl < 1e-11 and abs(dl - dlg) < 1e-13
    assert rel(C, Cg) < 1e-9 and rel(T, Tg) < 1e-9
    Co, To, _ = _oracle_steps(A, C0, T0, it)
    assert rel(C, Co) < 1e-9 and rel(T, To) < 1e-9
    # the oracle's delta over check_every steps at the stopping point
    Cp, _, _ = _oracle_steps(A, C0, T0, it - check_every)
    assert abs(dl - np.max(np.abs(o.spectrum(Co) - o.spectrum(Cp)))) < 1e-12


def test_absorb_mode_auto_selects_by_bond_dimension():
    """QRCTM_OPT_ABSORB_MODE = 2: layered from D = 6 up, explicit below -- bitwise the respective fixed mode."""
    for (d, D, chi, seed) in ((2, 6, 12, 3), (2, 4, 16, 2)):
        outs = {}
        for mode in (0, 1, 2):
            o_, _, _ = _one_step(d, D, chi, seed, absorb=mode)
            outs[mode] = o_
        same = 1 if D >= 6 else 0
        assert np.array_equal(outs[2]["T"], outs[same]["T"]) and np.array_equal(outs[2]["C"], outs[same]["C"])
        assert rel(outs[2]["T"], outs[1 - same]["T"]) < 1e-12


def test_large_chi_fallback_paths():
    """chi = 300 > 236: the corner spectrum takes the global-memory tridiagonalisation path; D = 1 keeps it cheap.
    Also a square c~ (m = chi) for the QR (19 panels, the last one ragged)."""
    d, D, chi = 2, 1, 300
    A, C0, T0 = gen_config(d, D, chi, 5)
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A); h.set_env(C0, T0)
    C, _ = h.get_env()
    assert np.max(np.abs(h.get_corner_spectrum() - o.spectrum(C))) < 5e-15 * chi
    h.step()
    a = o.build_a(A)
    Cr, Tr = o.normalize(C0, T0)
    s = o.qr_step(Cr, Tr, a)
    Co, To = o.normalize(s["Cn"], s["Tn"])
    Q, R = h.get_qr()
    assert np.linalg.norm(Q.T @ Q - np.eye(chi)) < chi * 2e-15 and rel(Q @ R, s["X"]) < 1e-13
    cond = np.linalg.cond(s["X"])
    C1, T1 = h.get_env()
    tol = max(1e-11, 1e-14 * cond)          # a square random c~ is ill-conditioned: Q is only determined to cond * eps
    assert rel(C1, Co) < tol and rel(T1, To) < tol
    it, dl = h.run(3, -1.0)
    assert it == 3 and np.isfinite(dl)
    h.close()


def test_odd_chi_and_d3_run_parity():
    """Odd chi (no 16-byte aligned rows: cp.async fallback GEMM, layered mode falls back to explicit) and d = 3."""
    d, D, chi = 3, 2, 9
    A, C0, T0 = gen_config(d, D, chi, 11)
    for absorb in (0, 1):
        h = pkg.QRCTM(d, D, chi)
        h.set_option(pkg.OPT_ABSORB_MODE, absorb)
        h.set_A(A); h.set_env(C0, T0)
        it, dl = h.run(12, -1.0)
        Co, To, a = _oracle_steps(A, C0, T0, 12)
        C, T = h.get_env()
        assert rel(C, Co) < 1e-10 and rel(T, To) < 1e-10
        assert abs(h.norm_per_site() / o.kappa(Co, To, a) - 1) < 1e-9
        h.close()


@pytest.mark.parametrize("d,D,chi,seed,steps", [(2, 2, 8, 0, 30), (2, 3, 20, 1, 10), (3, 2, 6, 4, 5), (2, 4, 32, 2, 3)])
def test_energy_nn_matches_oracle(d, D, chi, seed, steps):
    """NEXT-3: two-site RDM and bond energy from the GPU half network vs the oracle, same environment."""
    g = np.random.default_rng(seed + 100)
    A, C0, T0 = gen_config(d, D, chi, seed)
    H = g.standard_normal((d * d, d * d)); H = H + H.T
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A); h.set_env(C0, T0)
    h.run(steps, -1.0)
    C, T = h.get_env()
    e, rho = h.energy_nn(H, return_rho=True)
    rho_o = o.rdm2(C, T, A)
    assert rel(rho, rho_o) < 1e-11
    assert abs(e - o.energy_nn(C, T, A, H)) < 1e-10 * max(1.0, abs(e))
    assert abs(h.energy_nn(np.eye(d * d)) - 1.0) < 1e-12
    C2, T2 = h.get_env()
    assert np.array_equal(C, C2) and np.array_equal(T, T2)        # the environment is untouched
    h.step()                                                      # and the step still works afterwards
    h.close()


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3a", "cfg3b", "cfg4"])
def test_long_run_parity_at_baseline_iteration_counts(name):
    """BASELINE.json: cfg1 runs to tol 1e-10 or 500 iterations, cfg2 300, cfg3a/cfg3b 200 each, cfg4 100 iterations
    (cfg0's run: test_cfg0_*).  North-star bar for the run, on all five configs: relative error <= 1e-9 on the norm
    per site and on the top-10 normalised corner eigenvalues (iteration until convergence: PAPER.md:26)."""
    c = CONFIGS[name]
    A, C0, T0 = gen_config(c["d"], c["D"], c["chi"], c["seed"])
    a = o.build_a(A)
    h = pkg.QRCTM(c["d"], c["D"], c["chi"])
    h.set_A(A); h.set_env(C0, T0)
    it, dl = h.run(c["iters"], c["tol"])
    Co, To, ito, dlo, hist = o.run(C0, T0, a, "qr", c["iters"], c["tol"])
    assert abs(it - ito) <= 1
    if it != ito:                       # delta crossed tol one step apart: bring the oracle to the same count
        Co, To, _ = _oracle_steps(A, C0, T0, it)
    s, so = h.get_corner_spectrum(), o.spectrum(Co)
    assert np.max(np.abs(s[:10] - so[:10]) / so[:10]) < 1e-9
    k, ko = h.norm_per_site(), o.kappa(Co, To, a)
    assert abs(k / ko - 1) < 1e-9
    if it == c["iters"]:                # hit the cap (hazard H2 for cfg1's seed): deltas must agree too
        assert abs(dl - hist[-1]) <= 1e-9 * max(1.0, abs(hist[-1])) + 1e-12
    h.close()


def test_cfg4_five_iterations_run_parity():
    """The headline config through qrctm_run (graphs, overlapped check): 5 iterations against the oracle."""
    c = CONFIGS["cfg4"]
    A, C0, T0 = gen_config(c["d"], c["D"], c["chi"], c["seed"])
    h = pkg.QRCTM(c["d"], c["D"], c["chi"])
    h.set_A(A); h.set_env(C0, T0)
    it, dl = h.run(5, -1.0)
    assert it == 5
    Co, To, a = _oracle_steps(A, C0, T0, 5)
    C, T = h.get_env()
    assert rel(C, Co) < 1e-10 and rel(T, To) < 1e-10
    s, so = h.get_corner_spectrum(), o.spectrum(Co)
    assert np.max(np.abs(s[:10] - so[:10]) / so[:10]) < 1e-9
    so_prev = o.spectrum(_oracle_steps(A, C0, T0, 4)[0])
    assert abs(dl - np.max(np.abs(so - so_prev))) < 1e-12
    assert abs(h.norm_per_site() / o.kappa(Co, To, a) - 1) < 1e-9
    h.close()


def test_gemm_randomised_shapes_against_numpy():
    """40 random (M, N, K, transA) draws, ragged in every dimension, incl. views with odd leading dimensions:
    every tile configuration / split-K choice of the launcher gets exercised against NumPy."""
    g = np.random.default_rng(2024)
    import torch
    for trial in range(40):
        M = int(g.choice([1, 7, 33, 100, 129, 196, 500, 1025, 2401, 4000, 9604]))
        N = int(g.choice([1, 8, 49, 57, 98, 105, 196, 250, 1030, 2401]))
        K = int(g.choice([1, 3, 16, 49, 98, 196, 333, 1000, 2401]))
        if M * N * K > 6e9:
            K = 49
        transA = bool(g.integers(0, 2))
        padA, padB = int(g.integers(0, 3)), int(g.integers(0, 3))
        Afull = g.standard_normal((K, M + padA) if transA else (M, K + padA))
        Bfull = g.standard_normal((K, N + padB))
        Ad = torch_dev(Afull)[:, :M] if transA else torch_dev(Afull)[:, :K]
        Bd = torch_dev(Bfull)[:, :N]
        A = Afull[:, :M] if transA else Afull[:, :K]
        ref = (A.T if transA else A) @ Bfull[:, :N]
        out = pkg.gemm_f64(Ad, Bd, transA=transA).cpu().numpy()
        scale = np.linalg.norm(ref) if np.linalg.norm(ref) > 0 else 1.0
        assert np.linalg.norm(out - ref) / scale < 1e-13, (trial, M, N, K, transA, padA, padB)


@pytest.mark.parametrize("M,N,K", [
    (2000, 100, 4000),     # 16 tiles of 128x104, 250 k-tiles each: stream-K, every tile split over ~9 CTAs
    (9604, 196, 2401),     # K5's shape with a shorter K: 152 tiles on 148 CTAs
    (1100, 1030, 1500),    # 128x64 tiles, two CTAs per SM: 153 tiles on 296 CTAs, ragged in M, N and K
    (700, 260, 9000),      # 128x128 tiles (N pads least there), 18 tiles, K not a multiple of 16
    (4000, 196, 333),      # short K: split-K / plain tiles chosen by the cost model
    (3750, 150, 3750),     # K5 at cfg3b: one 160-wide tile column (128 x 160 tiles, warps of 64 x 40), stream-K
    (3000, 290, 700),      # two 160-wide tile columns, ragged in N
])
def test_gemm_k_splitting_schedules_against_numpy(M, N, K):
    """qrctm_gemm_f64_ws: with a scratch buffer the launcher may split K (split-K or stream-K).
    Result vs NumPy, bitwise reproducibility, and agreement with the unsplit schedule to summation-order rounding."""
    g = np.random.default_rng(M + 3 * N + 7 * K)
    A = g.standard_normal((K, M)); B = g.standard_normal((K, N))
    Ad, Bd = torch_dev(A), torch_dev(B)
    ref = A.T @ B
    out1 = pkg.gemm_f64(Ad, Bd, transA=True, work_bytes=256 << 20).cpu().numpy()
    out2 = pkg.gemm_f64(Ad, Bd, transA=True, work_bytes=256 << 20).cpu().numpy()
    plain = pkg.gemm_f64(Ad, Bd, transA=True).cpu().numpy()
    assert np.array_equal(out1, out2)
    assert rel(out1, ref) < 1e-13
    assert rel(out1, plain) < 1e-14
